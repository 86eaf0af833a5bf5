// fe_pipe.cu -- instantiations and launcher of the pipelined kernel (fe_pipe.cuh); a translation unit of its own so
// that it compiles in parallel with fengine.cu.
#include "fe_pipe.cuh"
#include "fe_plans.cuh"

namespace fe {

namespace {

template <int T, class Plan, bool F32OUT>
cudaError_t launch_one(const PipeParams &prm, int grid, bool set_attr, cudaStream_t stream)
{
    const size_t smem = PipeSmem<Plan>::bytes(prm.fir_warps);
    if (set_attr) {
        cudaError_t e = cudaFuncSetAttribute(pipe_kernel<T, Plan, F32OUT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    const int threads = Plan::tpf + 64 + 32 * prm.fir_warps;      // team + loader + flow + FIR warps
    pipe_kernel<T, Plan, F32OUT><<<grid, threads, smem, stream>>>(prm);
    return cudaGetLastError();
}

template <int T, bool F32OUT>
cudaError_t launch_n(int n, const PipeParams &prm, int grid, bool set_attr, cudaStream_t stream)
{
    switch (n) {
    case 1024: return launch_one<T, Plan2_1024, F32OUT>(prm, grid, set_attr, stream);
    case 2048: return launch_one<T, Plan2_2048, F32OUT>(prm, grid, set_attr, stream);
    case 4096: return launch_one<T, Plan2_4096, F32OUT>(prm, grid, set_attr, stream);
    case 8192: return launch_one<T, Plan2_8192, F32OUT>(prm, grid, set_attr, stream);
    }
    return cudaErrorInvalidValue;
}

template <bool F32OUT>
cudaError_t launch_T(int T, int n, const PipeParams &prm, int grid, bool set_attr, cudaStream_t stream)
{
    switch (T) {
    case 2: return launch_n<2, F32OUT>(n, prm, grid, set_attr, stream);
    case 4: return launch_n<4, F32OUT>(n, prm, grid, set_attr, stream);
    case 8: return launch_n<8, F32OUT>(n, prm, grid, set_attr, stream);
    case 16: return launch_n<16, F32OUT>(n, prm, grid, set_attr, stream);
    }
    return cudaErrorInvalidValue;
}

}  // namespace

int pipe_team_threads(int n) { return n >= 4096 ? Plan2_4096::tpf : Plan2_1024::tpf; }

size_t pipe_smem_bytes(int n, int fir_warps)
{
    switch (n) {
    case 1024: return PipeSmem<Plan2_1024>::bytes(fir_warps);
    case 2048: return PipeSmem<Plan2_2048>::bytes(fir_warps);
    case 4096: return PipeSmem<Plan2_4096>::bytes(fir_warps);
    case 8192: return PipeSmem<Plan2_8192>::bytes(fir_warps);
    }
    return 0;
}

cudaError_t pipe_launch(int T, int n, bool f32out, const PipeParams &prm, int grid, bool set_attr, cudaStream_t stream)
{
    return f32out ? launch_T<true>(T, n, prm, grid, set_attr, stream) : launch_T<false>(T, n, prm, grid, set_attr, stream);
}

}  // namespace fe
