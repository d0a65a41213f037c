// mvd_fft.cu -- FFT engine of libmvd (placeholder until the kernels land).
#include "mvd_internal.cuh"

int fft_supported(int, int) { return 0; }
int fft_setup(mvd_handle*, const float*) { return MVD_ERR_UNSUPPORTED; }
int fft_run(mvd_handle*, Workspace&, const uint16_t*, size_t, float*, int, cudaStream_t) { return MVD_ERR_UNSUPPORTED; }
int fft_default_chunk(const mvd_handle*) { return 1; }
