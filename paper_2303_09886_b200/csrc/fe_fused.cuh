// fe_fused.cuh -- the whole path (steps 1-7) as ONE persistent kernel for the pol-packed layout.
//
// Why.  The polyphase FIR wants to walk down the rows of a few columns (weights in registers),
// the FFT wants whole rows, so the FIR output g has to be transposed between the two.
// The paper's chain of kernels does that through device memory, which it identifies as the cost of its modular
// design.  Two kernels through HBM cost 8 bytes per real sample on top of the 2.25
// algorithmic ones; here the transposition goes through a small ring of scratch slots that
// stays resident in the 126 MB L2, so HBM sees only the packed input and the int8 output.
//
// How.  The call is cut into units u = (row chunk k, antenna a) of C spectra.  One grid of persistent CTAs
// draws tickets from a global counter; phase p of the ticket sequence holds
//     nb FIR tasks of unit p          (one block of tpf complex points = 2 tpf columns, C rows, both pols)
//     C  FFT tasks of unit p - LAG    (one spectrum, both pols)
// FIR task (u, b) writes rows of ring slot u mod D and bumps fir_done[u] (release); an FFT task of unit u waits
// (acquire) for fir_done[u] == nb, reads its row from L2, and bumps fft_done[u] as soon as the row is in
// registers / shared memory (after pass 1), which lets FIR tasks of unit u + D reuse the slot.  A task only ever
// waits for tasks with smaller tickets, which are already running on resident CTAs and never wait for larger
// ones, so the scheme cannot deadlock whatever the grid size.  FIR-heavy CTAs (FMA pipe) and FFT-heavy CTAs
// (shared memory, L2 latency) share each SM, which is where the overlap comes from.
#pragma once
#include "fe_common.cuh"
#include "fe_fft2.cuh"
#include "fe_fir2.cuh"

namespace fe {

struct FusedParams {
    Fir2Params fir;           // in, weights, coarse, n_coarse, stream_bytes, rows_in, lgN (g, m_*, chunk_cap unused)
    Fft2Params fft;           // out / out_f32, tables, delays, n_spectra, per_spectrum (g, m_*, chunk_cap unused)
    float *ring;              // D slots of C rows of n units of 16 bytes
    unsigned int *ctl;        // [0] ticket counter, [4, 4+U) fir_done, [4+U, 4+2U) fft_done; zeroed before the launch
    int64_t S;                // spectra per stream
    int A, C, D, LAG;         // antennas, rows per unit, ring slots, phases between a unit's FIR and FFT tasks
    int U;                    // units = ceil(S / C) * A, u = k * A + a
    int nb;                   // FIR tasks per unit = n / tpf
};

__device__ __forceinline__ void wait_counter(const unsigned int *ctr, unsigned int target, int tid)
{
    if (tid == 0) {
        while (ld_acquire_u32(ctr) < target) __nanosleep(64);
    }
    __syncthreads();
}

// Decode a ticket.  kind: 0 = nothing to do (padding of the sequence), 1 = FIR task, 2 = FFT task.
struct FusedTask {
    int kind, u, k, a, r;             // unit, chunk, antenna, column block (FIR) or row within the unit (FFT)
    const unsigned int *dep;          // counter this task waits for (null: none)
    unsigned int dep_target;
};

__device__ __forceinline__ FusedTask fused_decode(const FusedParams &prm, unsigned int ticket)
{
    FusedTask t;
    t.kind = 0;
    t.dep = nullptr;
    t.dep_target = 0;
    const unsigned int per_phase = (unsigned int)(prm.nb + prm.C);
    const int p = (int)(ticket / per_phase), r = (int)(ticket - (unsigned int)p * per_phase);
    const unsigned int *fir_done = prm.ctl + 4;
    const unsigned int *fft_done = prm.ctl + 4 + prm.U;
    t.u = t.k = t.a = t.r = 0;
    if (r < prm.nb) {
        if (p >= prm.U) return t;
        t.kind = 1;
        t.u = p;
        t.k = p / prm.A;
        t.a = p - t.k * prm.A;
        t.r = r;
        if (t.u >= prm.D) {                                // the slot's previous tenant has been read out
            const int up = t.u - prm.D, kp = up / prm.A;
            t.dep = fft_done + up;
            t.dep_target = (unsigned int)(min((int64_t)(kp + 1) * prm.C, prm.S) - (int64_t)kp * prm.C);
        }
    } else {
        const int u = p - prm.LAG;
        if (u < 0 || u >= prm.U) return t;
        const int k = u / prm.A;
        if ((int64_t)k * prm.C + (r - prm.nb) >= prm.S) return t;
        t.kind = 2;
        t.u = u;
        t.k = k;
        t.a = u - k * prm.A;
        t.r = r - prm.nb;
        t.dep = fir_done + u;
        t.dep_target = (unsigned int)prm.nb;
    }
    return t;
}

// Thread 0 draws the next ticket late in the current task (an FFT task: after pass 1; a FIR task: when its rows are
// written), samples the next task's dependency counter (acquire) after pass 2, and consumes both values only when
// the task ends, so the two round trips to L2 overlap the rest of the task.  The ticket is NOT drawn earlier than
// that: a CTA that sits on a ticket while it works through a long task delays everything that depends on it.
template <int T, class Plan, bool F32OUT>
__global__ void __launch_bounds__(Plan::tpf, (512 / Plan::tpf) > 0 ? (512 / Plan::tpf) : 1) fused2_kernel(const FusedParams prm)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ unsigned int s_ticket[2], s_ready[2];
    constexpr int n = Plan::n, N = 2 * n, tpf = Plan::tpf, warps = tpf / 32;
    static_assert((size_t)warps * kFirDepth * kFir2SlotBytes + 16 <= (size_t)Plan::units * 16, "FIR rings alias the FFT row buffer");
    const int tid = threadIdx.x;
    const int warp = tid >> 5;
    unsigned int *fir_done = prm.ctl + 4;
    unsigned int *fft_done = prm.ctl + 4 + prm.U;
    const unsigned int total = (unsigned int)(prm.U + prm.LAG) * (unsigned int)(prm.nb + prm.C);
    const size_t slot_floats = (size_t)prm.C * N * 2;
    const uint32_t ring_s = (uint32_t)__cvta_generic_to_shared(smem_raw + warp * kFirDepth * kFir2SlotBytes);

    if (tid == 0) {
        s_ticket[0] = atomicAdd(prm.ctl, 1u);
        s_ready[0] = 0;
    }
    for (int it = 0;; ++it) {
        __syncthreads();                                  // previous task is done with shared memory; ticket published
        const unsigned int ticket = s_ticket[it & 1];
        const bool ready = s_ready[it & 1] != 0;
        if (ticket >= total) break;
        unsigned int next_ticket = 0, next_seen = 0, next_target = 1;
        auto draw_next = [&] {
            if (tid == 0) asm volatile("atom.global.add.u32 %0, [%1], 1;" : "=r"(next_ticket) : "l"(prm.ctl) : "memory");
        };
        auto peek_next = [&] {                            // thread 0: sample the next task's dependency
            if (tid == 0) {
                next_target = 0;
                if (next_ticket < total) {
                    const FusedTask nt = fused_decode(prm, next_ticket);
                    if (nt.dep) {
                        next_target = nt.dep_target;
                        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(next_seen) : "l"(nt.dep) : "memory");
                    }
                }
            }
        };
        const FusedTask t = fused_decode(prm, ticket);

        if (t.kind == 1) {
            // ---------------- FIR task: unit u, column block r ----------------
            const int64_t row0 = (int64_t)t.k * prm.C;
            const int64_t m_stop = min(row0 + (int64_t)prm.C, prm.S);
            if (t.dep && !ready) wait_counter(t.dep, t.dep_target, tid);
            float *slot = prm.ring + (size_t)(t.u % prm.D) * slot_floats;
            const int i_pt = t.r * tpf + tid;
            const uint8_t *sbase = prm.fir.in + (int64_t)t.a * 2 * prm.fir.stream_bytes;
            const uint8_t *wsrc = sbase + (int64_t)(t.r * warps + warp) * kFir2SegBytes;
            const int32_t *ctab = prm.fir.coarse + (int64_t)t.a * 2 * prm.fir.n_coarse;
            int64_t m = row0;
            while (m < m_stop) {
                const int32_t c = ctab[prm.fir.n_coarse == 1 ? 0 : m];
                int64_t run_end = m_stop;
                if (prm.fir.n_coarse != 1) {
                    run_end = m + 1;
                    while (run_end < m_stop && ctab[run_end] == c) ++run_end;
                }
                float *grow0 = slot + (size_t)(m - row0) * N * 2;
                const int cr = (int)((int64_t)c & (int64_t)(N - 1));
                const bool mixed = (2 * i_pt + cr < N) && (2 * i_pt + 1 + cr >= N);
                if (__any_sync(0xffffffffu, mixed))
                    fir2_run<T, true>(prm.fir, wsrc, ring_s, (int64_t)c, m, (int)(run_end - m), i_pt, grow0);
                else
                    fir2_run<T, false>(prm.fir, wsrc, ring_s, (int64_t)c, m, (int)(run_end - m), i_pt, grow0);
                m = run_end;
            }
            draw_next();
            __threadfence();                              // this thread's rows are visible at L2 ...
            __syncthreads();                              // ... for every thread of the block ...
            if (tid == 0) red_release_add_u32(fir_done + t.u, 1u);   // ... before the unit counts this block
        } else if (t.kind == 2) {
            // ---------------- FFT task: unit u, row r ----------------
            const int64_t m = (int64_t)t.k * prm.C + t.r;
            if (!ready) wait_counter(t.dep, t.dep_target, tid);
            const float4 *grow = reinterpret_cast<const float4 *>(prm.ring + (size_t)(t.u % prm.D) * slot_floats + (size_t)t.r * N * 2);
            fft2_row<Plan, F32OUT>(prm.fft, grow, smem_raw, t.a, m, tid, [&] {
                if (tid == 0) red_release_add_u32(fft_done + t.u, 1u);      // the row has left the ring
                draw_next();
            }, peek_next);
        } else {
            draw_next();
        }
        if (tid == 0) {
            s_ticket[(it + 1) & 1] = next_ticket;
            s_ready[(it + 1) & 1] = next_seen >= next_target ? 1u : 0u;
        }
    }
}

}  // namespace fe
