// fe_split.cu -- instantiations and launchers of the split path (fe_split.cuh); a translation unit of its own so
// that it compiles in parallel with fengine.cu.
#include "fe_split.cuh"
#include "fe_plans.cuh"

namespace fe {

namespace {

template <int T, int K1, int M>
cudaError_t launch_fir_one(const SplitParams &prm, dim3 grid, bool set_attr, cudaStream_t stream)
{
    const size_t smem = split_producer_smem();
    if (set_attr) {
        cudaError_t e = cudaFuncSetAttribute(split_fir_kernel<T, K1, M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    split_fir_kernel<T, K1, M><<<grid, kSplitProducerThreads, smem, stream>>>(prm);
    return cudaGetLastError();
}

template <int K1, int M>
cudaError_t launch_fir_T(int T, const SplitParams &prm, dim3 grid, bool set_attr, cudaStream_t stream)
{
    switch (T) {
    case 2: return launch_fir_one<2, K1, M>(prm, grid, set_attr, stream);
    case 4: return launch_fir_one<4, K1, M>(prm, grid, set_attr, stream);
    case 8: return launch_fir_one<8, K1, M>(prm, grid, set_attr, stream);
    case 16: return launch_fir_one<16, K1, M>(prm, grid, set_attr, stream);
    }
    return cudaErrorInvalidValue;
}

template <class Plan, bool F32OUT>
cudaError_t launch_pair_one(const SplitParams &prm, dim3 grid, bool set_attr, cudaStream_t stream)
{
    using SM = SplitBigSmem<Plan>;
    if (set_attr) {
        cudaError_t e = cudaFuncSetAttribute(split_pair_kernel<Plan, 16, F32OUT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SM::bytes);
        if (e != cudaSuccess) return e;
    }
    split_pair_kernel<Plan, 16, F32OUT><<<grid, 2 * Plan::tpf, SM::bytes, stream>>>(prm);
    return cudaGetLastError();
}

template <int K1, bool F32OUT>
cudaError_t launch_fft_one(const SplitParams &prm, dim3 grid, bool set_attr, cudaStream_t stream)
{
    using SM = SplitFftSmem<K1>;
    if (set_attr) {
        cudaError_t e = cudaFuncSetAttribute(split_fft_kernel<K1, F32OUT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SM::bytes);
        if (e != cudaSuccess) return e;
    }
    split_fft_kernel<K1, F32OUT><<<grid, SM::warps * 32, SM::bytes, stream>>>(prm);
    return cudaGetLastError();
}

}  // namespace

bool split_supported(int n, int T) { return (n == 4096 || n == 16384 || n == 32768) && (T == 2 || T == 4 || T == 8 || T == 16); }
bool split_is_big(int n) { return n >= 16384; }

cudaError_t split_launch_fir(int T, int n, const SplitParams &prm, dim3 grid, bool set_attr, cudaStream_t stream)
{
    switch (n) {
    case 4096: return launch_fir_T<16, 256>(T, prm, grid, set_attr, stream);
    case 16384: return launch_fir_T<16, 1024>(T, prm, grid, set_attr, stream);
    case 32768: return launch_fir_T<16, 2048>(T, prm, grid, set_attr, stream);
    }
    return cudaErrorInvalidValue;
}

cudaError_t split_launch_fft(int n, bool f32out, const SplitParams &prm, dim3 grid, bool set_attr, cudaStream_t stream)
{
    switch (n) {
    case 4096:
        return f32out ? launch_fft_one<16, true>(prm, grid, set_attr, stream) : launch_fft_one<16, false>(prm, grid, set_attr, stream);
    case 16384:
        return f32out ? launch_pair_one<Plan2_1024, true>(prm, grid, set_attr, stream) : launch_pair_one<Plan2_1024, false>(prm, grid, set_attr, stream);
    case 32768:
        return f32out ? launch_pair_one<Plan2_2048, true>(prm, grid, set_attr, stream) : launch_pair_one<Plan2_2048, false>(prm, grid, set_attr, stream);
    }
    return cudaErrorInvalidValue;
}

}  // namespace fe
