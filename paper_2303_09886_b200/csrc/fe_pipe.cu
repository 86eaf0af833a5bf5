// fe_pipe.cu -- instantiations and launcher of the pipelined kernel (fe_pipe.cuh); a translation unit of its own so
// that it compiles in parallel with fengine.cu.
#include <mutex>

#include "fe_pipe.cuh"
#include "fe_plans.cuh"

namespace fe {

namespace {

// The dynamic shared-memory limit is an attribute of the FUNCTION (per device), not of a handle: it is raised here,
// never lowered, and remembered per instantiation and device, so that a second handle with fewer FIR warps cannot
// shrink it under the first.  The CTAs of the kernel spin-wait on one another (FIR warps of one CTA feed the FFT team of
// another), which is deadlock-free only when the whole grid is resident: the launch is a cooperative one, which the
// runtime refuses (cudaErrorCooperativeLaunchTooLarge) unless every CTA fits on the device at once and which is not
// started piecemeal beside kernels of other streams or handles.
template <int T, class Plan, bool F32OUT>
cudaError_t launch_one(const PipeParams &prm, int grid, bool /*set_attr*/, cudaStream_t stream)
{
    static std::mutex mu;
    static size_t limit_set[64] = {};
    const size_t smem = PipeSmem<Plan>::bytes(prm.fir_warps);
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    {
        std::lock_guard<std::mutex> lock(mu);
        if (smem > limit_set[dev]) {
            e = cudaFuncSetAttribute(pipe_kernel<T, Plan, F32OUT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
            limit_set[dev] = smem;
        }
    }
    const int threads = Plan::tpf + 64 + 32 * prm.fir_warps;      // team + loader + flow + FIR warps
    PipeParams arg = prm;
    void *args[] = {&arg};
    return cudaLaunchCooperativeKernel(reinterpret_cast<const void *>(&pipe_kernel<T, Plan, F32OUT>), dim3((unsigned)grid),
                                       dim3((unsigned)threads), args, smem, stream);
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
