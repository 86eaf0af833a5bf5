// fe_plans.cuh -- the compile-time FFT plans shared by the translation units.
#pragma once
#include "fe_fft.cuh"
#include "fe_fft2.cuh"

namespace fe {

// pol-sequential FFT (fe_fft.cuh): <n, passes, R1, R2, R3, R4, threads per pol-FFT, sweeps>
using Plan1024 = FftPlan<1024, 3, 8, 8, 16, 1, 64>;
using Plan2048 = FftPlan<2048, 3, 8, 16, 16, 1, 64>;
using Plan4096 = FftPlan<4096, 3, 16, 16, 16, 1, 128>;
using Plan8192 = FftPlan<8192, 4, 8, 8, 8, 16, 256>;
using Plan16384 = FftPlan<16384, 4, 16, 16, 8, 8, 512>;
using Plan32768 = FftPlan<32768, 4, 32, 16, 8, 8, 512, 2>;     // two sweeps of 16384 points

// pol-packed FFT (fe_fft2.cuh): <n, R2, R3, threads, sweeps>
using Plan2_1024 = Fft2Plan<1024, 8, 8, 128>;
using Plan2_2048 = Fft2Plan<2048, 8, 16, 128>;
using Plan2_4096 = Fft2Plan<4096, 16, 16, 256>;
using Plan2_8192 = Fft2Plan<8192, 16, 16, 256, 2>;    // two sweeps of 4096 points

// launcher of the persistent pol-packed FFT kernel (fe_fft2p.cu)
bool fft2p_supported(int n);
cudaError_t fft2p_launch(int n, bool f32out, const Fft2Params &prm, int A, int grid, bool set_attr, cudaStream_t stream);

// launcher of the pipelined kernel (fe_pipe.cu)
struct PipeParams;
int pipe_team_threads(int n);
size_t pipe_smem_bytes(int n, int fir_warps);
cudaError_t pipe_launch(int T, int n, bool f32out, const PipeParams &prm, int grid, bool set_attr, cudaStream_t stream);

}  // namespace fe
