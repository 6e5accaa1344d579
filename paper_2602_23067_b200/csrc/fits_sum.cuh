// fits_sum.cuh -- DATASUM reduction kernel (fits_sum.cu), host-side launch interface.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

// *d_acc += (sum of the big-endian 32-bit words of d_data[0, nbytes), tail bytes zero-extended), kept
// modulo 2^32 - 1 in a 64-bit accumulator; d_data 16-byte aligned.  Enqueued on `s`, no synchronisation.
cudaError_t launch_fits_sum32(const uint8_t *d_data, uint64_t nbytes, unsigned long long *d_acc, int sm_count,
                              cudaStream_t s);
// end-around-carry fold of the accumulator to the 32-bit 1's-complement sum
uint32_t fits_sum_fold(unsigned long long s);
