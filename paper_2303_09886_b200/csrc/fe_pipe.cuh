// fe_pipe.cuh -- the whole path (steps 1-7) as ONE persistent, warp-specialised kernel for the
// pol-packed layout: the FIR of Eq. (1) feeds the FFT through a small ring that stays in L2, so the FP32 intermediate
// never goes to HBM (BASELINE.json north_star (d); the paper's own conclusion: "modular design does
// not work well for memory-bound applications").
//
// Why a ring at all.  The polyphase FIR wants to walk down the rows of a few columns with its weights and T partial
// sums in registers; one row of one antenna (N columns, both pols) is 48 N registers of such
// state, more than six SMs' register files at N = 8192.  The FFT wants whole rows in one SM's shared memory.  The
// transposition between the two is therefore an exchange between SMs, and on B200 the L2 (about 40 B/clk/SM) is the
// widest path for it.  What the round-1 ticket kernel got wrong is fixed here:
//   * FIR state persists: a FIR warp owns 32 complex points (64 columns) of one "track" and walks down a whole
//     segment of an antenna's spectra (a "job") without ever restarting, so the T - 1 warm-up rows are paid once
//     per job instead of once per 64-row unit;
//   * roles run concurrently inside every CTA: FIR warps (FMA pipe, almost no shared memory) next to an FFT team
//     (shared memory, barriers) next to one loader lane, and they synchronise through mbarriers and named barriers,
//     never through a CTA-wide __syncthreads or a spin in a warp that also computes;
//   * rows come out of the ring by bulk copy (TMA, cp.async.bulk) into a landing buffer while the team transforms
//     the previous row, so pass 1 of the FFT reads shared memory instead of waiting on 16 dependent L2 loads;
//   * the ring is a few rows per track (default 32 rows = 16 MB at n = 4096) instead of whole 64-row units.
//
// Work decomposition.  The call's A antennas x S spectra are cut into n_jobs = A * K jobs (antenna a, segment k of
// Sseg spectra).  J tracks run concurrently; track t runs the jobs t, t + J, t + 2J, ... one after the other.  A track
// is served by wpj = n / 32 FIR warps (each a fixed run of 32 complex points), spread over the CTAs.  Rows of a track
// get consecutive sequence numbers (jobs padded to whole groups of G = 8 rows) and live in ring slot seq mod D.
//
// Ordering.  FFT work is handed out by a global ticket counter in production order (group p of every track, then
// group p + 1, ...).  ready[t][p] counts the FIR warps that have stored group p (target wpj); freed[t][p] counts
// the rows of group p that have left the ring (target G; padding rows are counted by whoever draws their ticket).  A
// FIR warp may overwrite group p - D/G's slots only when freed[..] says so.  Every wait is on work with a smaller
// ticket / an earlier group, which is owned by a CTA that is already running, so the scheme cannot deadlock as long
// as all CTAs are resident (grid <= number of SMs, one CTA per SM).
#pragma once
#include "fe_common.cuh"
#include "fe_fft2.cuh"
#include "fe_fir2.cuh"

namespace fe {

constexpr int kPipeG = 8;                 // rows per signalling group (half an unrolled FIR block)
constexpr int kPipeCtlHeader = 64;        // control words before the counters ([0] = ticket counter)
constexpr int kPipeMaxThreads = 480;          // 15 warps: 136 registers per thread, which the FIR loop needs to stay out of local memory

struct PipeParams {
    Fir2Params fir;           // in, weights, coarse, n_coarse, stream_bytes, rows_in, lgN (g, m_*, chunk_cap unused)
    Fft2Params fft;           // out / out_f32, tables, delays, n_spectra, per_spectrum (g, m_*, chunk_cap unused)
    float *ring;              // [J][D] rows of n units of 16 bytes
    unsigned int *ctl;        // [0] ticket; ready[t][x] at 64 + t*GP + x; freed[t][x] at 64 + (J + t)*GP + x
    int64_t m_lo, S;          // this launch transforms the spectra [m_lo, m_lo + S) of the call
    int A, K, Sseg;           // antennas, segments per antenna, spectra per segment (the last one may be shorter)
    int J, wpj;               // tracks, FIR warps per track
    int D, GP;                // ring rows per track (power of two, multiple of G), groups per track (counter pitch)
    int fir_warps;            // FIR warps per CTA
    unsigned int total_tickets;
    unsigned long long *stats;  // optional (option "pipe_stats"): 16 clock counters per CTA, see kPipeStat*
};

// per-CTA clock counters (SM clocks) of the optional statistics
enum { kStTeamWaitFull, kStTeamRow, kStTeamRows, kStLoadWaitEmpty, kStLoadWaitReady, kStLoadWaitLand, kStLoadRows,
       kStFirSpin, kStFirTotal, kStFirSteps, kStTeamTotal, kStCount = 16 };

// job j = (segment k = j / A, antenna a = j % A); spectra m_lo + [k * Sseg, min(S, (k + 1) * Sseg))
struct PipeJob {
    int a, m_begin, len, n_groups;
};
__device__ __forceinline__ PipeJob pipe_job(const PipeParams &prm, int j)
{
    PipeJob jb;
    const int k = j / prm.A;
    jb.a = j - k * prm.A;
    jb.len = (int)min((int64_t)prm.Sseg, prm.S - (int64_t)k * prm.Sseg);
    jb.m_begin = (int)prm.m_lo + k * prm.Sseg;
    jb.n_groups = (jb.len + kPipeG - 1) / kPipeG;
    return jb;
}

// ---- FIR role: the sink that puts finished rows into the ring (see Fir2ScratchSink for the protocol) ------------
// The FIR loop lives at the register limit (64 partial sums + 32 weights per thread) and must never execute a
// device-scope fence: MEMBAR.GPU waits for everything the warp has in flight, including the cp.async prefetch of
// input rows that are still on their way from HBM (measured: with a release per 8 rows in the FIR warps a step took
// 1100 clocks instead of 250).  So a FIR warp talks to shared memory only: it publishes how many groups of its
// track it has stored (PROG) and reads how many it may store (LIMIT); the flow warp of the CTA (below) turns PROG
// into device-scope releases of the ready counters and the freed counters into LIMIT.  Both numbers count groups of
// the track from its first job on and only ever grow, so job boundaries need no handshake.
// Registers: only what every step needs (sp, n_out, seq_run, base_off); the rest sits in the warp's 32-byte record.
template <int T, int N>
struct PipeSink {
    const PipeParams &prm;            // __grid_constant__ kernel parameter (constant bank)
    uint32_t ws;                      // shared-space address of this warp's record
    uint32_t base_off;                // byte offset of this thread's unit in slot 0 of its track's ring
    int n_out, sp;                    // per run
    unsigned int seq_run;             // sequence number of the run's row 0
    static constexpr uint32_t row_bytes = (uint32_t)N * 8u;
    enum { F_PROG, F_LIMIT, F_GBASE, F_JOB_LEN, F_RUN_OFF, F_JOB };

    __device__ __forceinline__ int ld(int field) const
    {
        int v;
        asm volatile("ld.volatile.shared.s32 %0, [%1];" : "=r"(v) : "r"(ws + 4u * field) : "memory");
        return v;
    }
    __device__ __forceinline__ void st(int field, int v) const { asm volatile("st.volatile.shared.s32 [%0], %1;" ::"r"(ws + 4u * field), "r"(v) : "memory"); }

    __device__ __forceinline__ void begin_run(int lag, int, int n_out_)
    {
        sp = lag - T;
        n_out = n_out_;
        seq_run = (unsigned int)(ld(F_GBASE) * kPipeG + ld(F_RUN_OFF));
    }
    __device__ __forceinline__ void store(float4 cur)
    {
        const unsigned int slot = (seq_run + (unsigned int)sp) & (unsigned int)(prm.D - 1);
        const unsigned char *dst = reinterpret_cast<const unsigned char *>(prm.ring) + ((size_t)slot * row_bytes + base_off);
        asm volatile("{\n\t.reg .pred p;\n\tsetp.lt.u32 p, %5, %6;\n\t@p st.global.v4.f32 [%0], {%1, %2, %3, %4};\n\t}"
                     ::"l"(dst), "f"(cur.x), "f"(cur.y), "f"(cur.z), "f"(cur.w), "r"((unsigned)sp), "r"((unsigned)n_out) : "memory");
        ++sp;
    }
    // every lane of the warp has stored the track's groups below `abs`
    __device__ __forceinline__ void publish(int abs) const
    {
        if (abs > ld(F_PROG)) {
            __syncwarp();
            if ((threadIdx.x & 31) == 0) {
                __threadfence_block();                 // the lanes' rows before the progress word (CTA scope: cheap)
                st(F_PROG, abs);
            }
            __syncwarp();
        }
    }
    // steps s .. s + 7 store run rows up to s + 8 - T (a lagging column is one row ahead): their slots must be free
    __device__ __forceinline__ void before_steps(int s)
    {
        const int need_row = min(ld(F_RUN_OFF) + min(s + 8 - T, n_out - 1), ld(F_JOB_LEN) - 1);
        if (need_row < 0) return;
        const int need = ld(F_GBASE) + need_row / kPipeG + 1;
        if (ld(F_LIMIT) >= need) return;
        const long long t0 = clock64();
        while (ld(F_LIMIT) < need) __nanosleep(20);
        if (prm.stats && (threadIdx.x & 31) == 0) atomicAdd(prm.stats + (size_t)blockIdx.x * kStCount + kStFirSpin, (unsigned long long)(clock64() - t0));
    }
    // after step s every lane has stored the run rows <= s - T
    __device__ __forceinline__ void after_steps(int s)
    {
        const int done = ld(F_RUN_OFF) + min(max(s - T + 1, 0), n_out);
        publish(ld(F_GBASE) + done / kPipeG);
    }
    __device__ __forceinline__ void end_run()
    {
        const int done = ld(F_RUN_OFF) + n_out, job_len = ld(F_JOB_LEN);
        publish(ld(F_GBASE) + (done >= job_len ? (job_len + kPipeG - 1) / kPipeG : done / kPipeG));
    }
};

__device__ __forceinline__ unsigned int ld_relaxed_u32(const unsigned int *p)
{
    unsigned int v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

template <class Plan>
struct PipeSmem {
    static constexpr int NS = Plan::n <= 4096 ? 2 : 1;                        // landing buffers
    static constexpr uint32_t row_bytes = (uint32_t)Plan::n * 16u;
    static constexpr uint32_t sph_off = (uint32_t)Plan::units * 16u;
    static constexpr uint32_t l_off = (sph_off + (uint32_t)sizeof(SpectrumPhase2) + 127u) & ~127u;
    static constexpr uint32_t bar_off = l_off + NS * row_bytes;              // full[2], empty[2] (8 B each), meta[2] (16 B each)
    static constexpr uint32_t fir_off = bar_off + 64u;
    static constexpr uint32_t fir_ring = (uint32_t)(kFirDepth * kFir2SlotBytes) + 32u;     // input ring + PipeWarpState
    __host__ __device__ static constexpr size_t bytes(int fir_warps) { return (size_t)fir_off + (size_t)fir_warps * fir_ring + 16; }
};

template <int T, class Plan, bool F32OUT>
__global__ void __launch_bounds__(kPipeMaxThreads, 1) pipe_kernel(const __grid_constant__ PipeParams prm)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    using SM = PipeSmem<Plan>;
    constexpr int NS = SM::NS, G = kPipeG, tpf = Plan::tpf, team_warps = tpf / 32;
    constexpr int N = 2 * Plan::n;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t s_base = smem_u32(smem_raw);
    const uint32_t full0 = s_base + SM::bar_off, empty0 = full0 + 16, meta0 = full0 + 32;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, 1);
        }
        mbar_fence_init();
    }
    if (tid < prm.fir_warps * 8)                          // PROG = LIMIT = 0 in every FIR warp's record
        reinterpret_cast<int *>(smem_raw + SM::fir_off + (size_t)(tid >> 3) * SM::fir_ring + kFirDepth * kFir2SlotBytes)[tid & 7] = 0;
    __syncthreads();                                      // the only CTA-wide barrier: roles part here

    unsigned int *const ready_all = prm.ctl + kPipeCtlHeader;
    unsigned int *const freed_all = ready_all + (size_t)prm.J * prm.GP;
    const size_t row_floats = (size_t)N * 2;

    if (warp < team_warps) {
        // ================= FFT team: one spectrum (both pols) at a time out of the landing buffers =================
        const auto sync = [] { bar_sync(1, tpf); };
        for (unsigned int it = 0;; ++it) {
            const int st = (int)(it % NS);
            const long long t0 = prm.stats ? clock64() : 0;
            mbar_wait(full0 + 8 * st, (it / NS) & 1u);
            const long long t1 = prm.stats ? clock64() : 0;
            int4 md;
            asm volatile("ld.shared.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(md.x), "=r"(md.y), "=r"(md.z), "=r"(md.w) : "r"(meta0 + 16 * st) : "memory");
            if (md.w) break;                              // no more tickets
            const RowInShared row{s_base + SM::l_off + (uint32_t)st * SM::row_bytes};
            fft2_row<Plan, F32OUT>(prm.fft, row, smem_raw, md.x, (int64_t)md.y, tid, sync, [&] {
                if (tid == 0) mbar_arrive(empty0 + 8 * st);              // the landing buffer may be refilled
            });
            sync();                                       // exchange buffer and phasors are reused by the next row
            if (prm.stats && tid == 0) {
                unsigned long long *st_ = prm.stats + (size_t)blockIdx.x * kStCount;
                st_[kStTeamWaitFull] += (unsigned long long)(t1 - t0);
                st_[kStTeamRow] += (unsigned long long)(clock64() - t1);
                st_[kStTeamRows] += 1;
            }
        }
    } else if (warp == team_warps) {
        // ================= loader: tickets, dependencies, bulk copies =================
        if (lane != 0) return;
        const unsigned int per = (unsigned int)(prm.J * G);
        unsigned int it = 0;
        for (;;) {
            const unsigned int t = atomicAdd(prm.ctl, 1u);
            if (t >= prm.total_tickets) break;
            const int p = (int)(t / per);
            const int rem = (int)(t - (unsigned int)p * per);
            const int track = rem / G, i = rem - track * G;
            // the job of this track that group p belongs to
            PipeJob jb{};
            int gbase = 0;
            bool found = false;
            for (int j = track; j < prm.A * prm.K; j += prm.J) {
                jb = pipe_job(prm, j);
                if (p < gbase + jb.n_groups) {
                    found = true;
                    break;
                }
                gbase += jb.n_groups;
            }
            if (!found) continue;                         // this track has fewer groups than the longest one
            const int row = (p - gbase) * G + i;
            const int cidx = track * prm.GP + p;
            if (row >= jb.len) {                          // padding of the job's last group: nothing to load
                red_release_add_u32(freed_all + cidx, 1u);
                continue;
            }
            const int st = (int)(it % NS);
            const long long t0 = prm.stats ? clock64() : 0;
            mbar_wait(empty0 + 8 * st, ((it / NS) & 1u) ^ 1u);
            const long long t1 = prm.stats ? clock64() : 0;
            {
                // polled at L2 without the L1 invalidation an acquire load carries; one acquire once the count is there
                const unsigned int *r = ready_all + cidx;
                while (ld_relaxed_u32(r) < (unsigned int)prm.wpj) __nanosleep(64);
                (void)ld_acquire_u32(r);
            }
            fence_proxy_async();
            const long long t2 = prm.stats ? clock64() : 0;
            asm volatile("st.shared.v4.s32 [%0], {%1,%2,%3,%4};" ::"r"(meta0 + 16 * st), "r"(jb.a), "r"(jb.m_begin + row), "r"(cidx), "r"(0) : "memory");
            mbar_arrive_expect_tx(full0 + 8 * st, SM::row_bytes);
            const unsigned int slot = (unsigned int)(p * G + i) & (unsigned int)(prm.D - 1);
            const unsigned char *src = reinterpret_cast<const unsigned char *>(prm.ring + ((size_t)track * prm.D + slot) * row_floats);
            const uint32_t dst = s_base + SM::l_off + (uint32_t)st * SM::row_bytes;
            constexpr uint32_t chunk = 16384;
#pragma unroll 1
            for (uint32_t off = 0; off < SM::row_bytes; off += chunk) bulk_g2s(dst + off, src + off, chunk, full0 + 8 * st);
            mbar_wait(full0 + 8 * st, (it / NS) & 1u);    // the row has landed, i.e. left the ring: its slot may be reused
            red_release_add_u32(freed_all + cidx, 1u);
            if (prm.stats) {
                unsigned long long *st_ = prm.stats + (size_t)blockIdx.x * kStCount;
                st_[kStLoadWaitEmpty] += (unsigned long long)(t1 - t0);
                st_[kStLoadWaitReady] += (unsigned long long)(t2 - t1);
                st_[kStLoadWaitLand] += (unsigned long long)(clock64() - t2);
                st_[kStLoadRows] += 1;
            }
            ++it;
        }
        const int st = (int)(it % NS);
        mbar_wait(empty0 + 8 * st, ((it / NS) & 1u) ^ 1u);
        asm volatile("st.shared.v4.s32 [%0], {%1,%1,%1,%2};" ::"r"(meta0 + 16 * st), "r"(0), "r"(1) : "memory");
        mbar_arrive(full0 + 8 * st);
    } else if (warp == team_warps + 1) {
        // ================= flow warp: lane l serves FIR warp l of this CTA =================
        // PROG (shared) -> ready counters (device scope, release): the fence is paid here, not in the FIR warps.
        // freed counters -> LIMIT (shared): how far the FIR warp may run ahead of the FFT teams.
        const int gw = (int)blockIdx.x * prm.fir_warps + lane;
        const bool active = lane < prm.fir_warps && gw < prm.J * prm.wpj;
        const int track = active ? gw / prm.wpj : 0;
        int total = 0;                                    // groups of the track
        if (active)
            for (int j = track; j < prm.A * prm.K; j += prm.J) total += pipe_job(prm, j).n_groups;
        const uint32_t ws = s_base + SM::fir_off + (uint32_t)lane * SM::fir_ring + (uint32_t)(kFirDepth * kFir2SlotBytes);
        unsigned int *ready = ready_all + (size_t)track * prm.GP;
        const unsigned int *freed = freed_all + (size_t)track * prm.GP;
        const int DG = prm.D / G;
        int sent = 0, granted = 0;
        for (;;) {
            int prog = 0;
            if (active) asm volatile("ld.volatile.shared.s32 %0, [%1];" : "=r"(prog) : "r"(ws) : "memory");
            const bool news = prog > sent;
            if (__any_sync(0xffffffffu, news)) {
                fence_proxy_async();                      // the rows are read by bulk copies (async proxy)
                if (news) {
#pragma unroll 1
                    for (int x = sent; x < prog; ++x) red_release_add_u32(ready + x, 1u);
                    sent = prog;
                }
            }
            if (active && granted < total) {
                int g = granted;
                while (g < total && (g < DG || ld_relaxed_u32(freed + (g - DG)) >= (unsigned int)G)) ++g;
                if (g != granted) {
                    granted = g;
                    asm volatile("st.volatile.shared.s32 [%0], %1;" ::"r"(ws + 4u), "r"(g) : "memory");
                }
            }
            if (__all_sync(0xffffffffu, !active || sent >= total)) break;
            __nanosleep(100);
        }
    } else {
        // ================= FIR warps: a fixed run of 32 complex points of one track, job after job =================
        const int fw = warp - team_warps - 2;
        if (fw >= prm.fir_warps || (int)blockIdx.x * prm.fir_warps + fw >= prm.J * prm.wpj) return;
        const uint32_t ring_s = s_base + SM::fir_off + (uint32_t)fw * SM::fir_ring;
        using Sink = PipeSink<T, N>;
        // Everything that outlives a run (which job, which spectrum comes next) sits in the warp's shared-memory
        // record and is re-read here, so that no loop-carried value competes with the FIR loop for registers.
        if (lane == 0) {
            const int track0 = ((int)blockIdx.x * prm.fir_warps + fw) / prm.wpj;
            Sink s0{prm, ring_s + (uint32_t)(kFirDepth * kFir2SlotBytes), 0u, 0, 0, 0u};
            s0.st(Sink::F_JOB, track0);
            s0.st(Sink::F_GBASE, 0);
            s0.st(Sink::F_RUN_OFF, 0);
            const long long t = clock64();
            s0.st(6, (int)(t & 0xffffffffll));
            s0.st(7, (int)(t >> 32));
        }
        __syncwarp();
        for (;;) {
            Sink sink{prm, ring_s + (uint32_t)(kFirDepth * kFir2SlotBytes), 0u, 0, 0, 0u};
            const int j = sink.ld(Sink::F_JOB);
            if (j >= prm.A * prm.K) break;
            const int gw = (int)blockIdx.x * prm.fir_warps + fw;
            const int track = gw / prm.wpj, q = gw - track * prm.wpj;
            const int i_pt = q * 32 + lane;
            sink.base_off = (uint32_t)(((size_t)track * prm.D * row_floats + 4 * (size_t)i_pt) * sizeof(float));
            const PipeJob jb = pipe_job(prm, j);
            const int run_off = sink.ld(Sink::F_RUN_OFF);
            const uint8_t *wsrc = prm.fir.in + (int64_t)jb.a * 2 * prm.fir.stream_bytes + (int64_t)q * kFir2SegBytes;
            const int32_t *ctab = prm.fir.coarse + (int64_t)jb.a * 2 * prm.fir.n_coarse;
            const int64_t m = (int64_t)jb.m_begin + run_off, m_stop = (int64_t)jb.m_begin + jb.len;
            const int32_t c = ctab[prm.fir.n_coarse == 1 ? 0 : m];
            int64_t run_end = m_stop;
            if (prm.fir.n_coarse != 1) {
                run_end = m + 1;
                while (run_end < m_stop && ctab[run_end] == c) ++run_end;
            }
            __syncwarp();
            if (lane == 0) sink.st(Sink::F_JOB_LEN, jb.len);
            __syncwarp();
            const int cr = (int)((int64_t)c & (int64_t)(N - 1));
            const bool mixed = (2 * i_pt + cr < N) && (2 * i_pt + 1 + cr >= N);
            const int n_run = (int)(run_end - m);
            if (__any_sync(0xffffffffu, mixed))
                fir2_run<T, true, Sink, N>(prm.fir, wsrc, ring_s, (int64_t)c, m, n_run, i_pt, sink);
            else
                fir2_run<T, false, Sink, N>(prm.fir, wsrc, ring_s, (int64_t)c, m, n_run, i_pt, sink);
            __syncwarp();
            if (lane == 0) {                              // what comes next: the rest of this job, or the track's next job
                const int ro = sink.ld(Sink::F_RUN_OFF) + sink.n_out, len = sink.ld(Sink::F_JOB_LEN);
                if (ro < len) {
                    sink.st(Sink::F_RUN_OFF, ro);
                } else {
                    sink.st(Sink::F_RUN_OFF, 0);
                    sink.st(Sink::F_GBASE, sink.ld(Sink::F_GBASE) + (len + G - 1) / G);
                    sink.st(Sink::F_JOB, sink.ld(Sink::F_JOB) + prm.J);
                }
            }
            __syncwarp();
        }
        if (prm.stats && lane == 0) {
            Sink s1{prm, ring_s + (uint32_t)(kFirDepth * kFir2SlotBytes), 0u, 0, 0, 0u};
            const long long t_start = (long long)(((unsigned long long)(unsigned int)s1.ld(7) << 32) | (unsigned int)s1.ld(6));
            atomicAdd(prm.stats + (size_t)blockIdx.x * kStCount + kStFirTotal, (unsigned long long)(clock64() - t_start));
            atomicAdd(prm.stats + (size_t)blockIdx.x * kStCount + kStFirSteps, 1ull);
        }
    }
}

}  // namespace fe
