// Internal launch interface between west.cu and fft_dense.cu (dense C2C 3D FFT, Fig. 3 of the paper).
#pragma once
#include <cuda_runtime.h>

bool west_dense_fft_supported(int n);
// tw: device table of n complex<double>, tw[m] = exp(+2 pi i m / n).  in == out allowed.  Three launches on stm.
cudaError_t west_dense_fft3d(int n, int f32, int sign, int n_batch, cudaStream_t stm, const void* in, void* out, const void* tw);
