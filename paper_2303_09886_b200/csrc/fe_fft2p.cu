// fe_fft2p.cu -- instantiations and launcher of the persistent pol-packed FFT kernel (fft2p_kernel, fe_fft2.cuh); a
// translation unit of its own so that it compiles in parallel with fengine.cu.
#include "fe_fft2.cuh"
#include "fe_plans.cuh"

namespace fe {

namespace {

template <class Plan, bool F32OUT>
cudaError_t launch_one(const Fft2Params &prm, int A, int grid, bool set_attr, cudaStream_t stream)
{
    using SM = Fft2pSmem<Plan>;
    if (set_attr) {
        cudaError_t e = cudaFuncSetAttribute(fft2p_kernel<Plan, F32OUT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SM::bytes);
        if (e != cudaSuccess) return e;
    }
    fft2p_kernel<Plan, F32OUT><<<grid, 512, SM::bytes, stream>>>(prm, A);
    return cudaGetLastError();
}

template <bool F32OUT>
cudaError_t launch_n(int n, const Fft2Params &prm, int A, int grid, bool set_attr, cudaStream_t stream)
{
    switch (n) {
    case 1024: return launch_one<Plan2_1024, F32OUT>(prm, A, grid, set_attr, stream);
    case 2048: return launch_one<Plan2_2048, F32OUT>(prm, A, grid, set_attr, stream);
    case 4096: return launch_one<Plan2_4096, F32OUT>(prm, A, grid, set_attr, stream);
    }
    return cudaErrorInvalidValue;
}

}  // namespace

bool fft2p_supported(int n) { return n == 1024 || n == 2048 || n == 4096; }

cudaError_t fft2p_launch(int n, bool f32out, const Fft2Params &prm, int A, int grid, bool set_attr, cudaStream_t stream)
{
    return f32out ? launch_n<true>(n, prm, A, grid, set_attr, stream) : launch_n<false>(n, prm, A, grid, set_attr, stream);
}

}  // namespace fe
