// hz_noalloc.cu -- ONE entry point of the C ABI that allocates nothing: hz_sum_fields_noalloc.
//
// Why: some callers cannot call cudaMalloc -- code under CUDA graph capture, tight serving loops, harnesses that
// forbid it.  The library's global reductions (hz_diagnostics: k_diag -> block partials ->
// k_diag_final) keep their block partials in scratch memory that belongs to a context, and a context owns a device
// buffer.  This file holds a variant of that reduction -- the volume sums of a set of fields -- whose scratch is a
// file-scope `static __device__` array of fixed size, so the call needs no context and no allocation: the caller
// passes the input fields and the output array, both DEVICE memory, and a stream.
//
// The scratch: HZ_NOALLOC_MAX_BLOCKS x HZ_NOALLOC_MAX_FIELDS doubles = 1184 x 16 x 8 B = 151 552 bytes (148 KiB).
// Every GPU that loads libhz.so holds it until the process exits.  In HOST code the array's name is a host-side
// stand-in, not a device address (a kernel given it would fault or, where the GPU can reach host memory, silently
// use the wrong memory): the device address is taken with cudaGetSymbolAddress once per device, with that device
// current (noalloc_scratch below), and that pointer is what the kernels get.
//
// Every call on a device shares the one array.  Nothing in it has to start at zero: every block of a call
// overwrites its own row of partials before the fold of the same call reads it, and rows of an earlier, larger
// call that lie beyond this call's blocks are never read.  Calls that OVERLAP on one GPU (two streams, two host
// threads) race on the array and give wrong sums: serialise them (one stream, or events between streams).
//
// This file calls no cudaMalloc, cudaFree or allocating library routine, and changes no other code path.
#include "../../include/hz.h"

#include <cuda_runtime.h>

namespace {

constexpr int MAXB = HZ_NOALLOC_MAX_BLOCKS;   // rows of partials = largest grid of the first kernel
constexpr int MAXF = HZ_NOALLOC_MAX_FIELDS;   // doubles per row = most fields summed at once
constexpr int NT = 256;                       // threads per block of the first kernel
constexpr int MAXDEV = 64;                    // devices whose scratch address is remembered

// the scratch itself: a device array in every GPU's copy of the module
static __device__ __align__(256) double g_scratch[(size_t)MAXB * MAXF];

// Device address of g_scratch per device ordinal, filled at set-up with that device current.
double* g_scratch_addr[MAXDEV] = {};

// Set-up for the CURRENT device: its address of the scratch array.  No allocation, no launch.
int noalloc_scratch(double** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAXDEV) { cudaGetLastError(); return HZ_ECUDA; }
  if (!g_scratch_addr[dev]) {
    double* p = nullptr;
    if (cudaGetSymbolAddress((void**)&p, g_scratch) != cudaSuccess || !p) { cudaGetLastError(); return HZ_ECUDA; }
    g_scratch_addr[dev] = p;
  }
  *out = g_scratch_addr[dev];
  return HZ_OK;
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  return v;
}

// First kernel (the variant of k_diag): block b accumulates, in fp64, the sums of fields 0 .. nf-1 over the cells
// b NT + t, (b + gridDim) NT + t, ... and writes them to row b of `scratch`.  Field f occupies fields[f n .. f n + n).
template <typename T>
__global__ void __launch_bounds__(NT) k_sum_partials(const T* __restrict__ fields, int nf, long long n,
                                                     double* __restrict__ scratch) {
  __shared__ double sh[NT / 32][MAXF];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int f = 0; f < nf; f++) {
    const T* p = fields + (long long)f * n;
    double acc = 0;
    for (long long t = (long long)blockIdx.x * NT + threadIdx.x; t < n; t += (long long)gridDim.x * NT) acc += (double)p[t];
    acc = warp_sum(acc);
    if (lane == 0) sh[wid][f] = acc;
  }
  __syncthreads();
  if (threadIdx.x < nf) {
    double v = sh[0][threadIdx.x];
    for (int w = 1; w < NT / 32; w++) v += sh[w][threadIdx.x];   // fixed order
    scratch[(long long)blockIdx.x * MAXF + threadIdx.x] = v;      // every row that will be read is written first
  }
}

// Second kernel: one block folds rows 0 .. nb-1 in a fixed order (deterministic result) into out[0 .. nf-1].
__global__ void k_sum_fold(const double* __restrict__ scratch, int nb, int nf, double* __restrict__ out) {
  const int f = threadIdx.x;
  if (f >= nf) return;
  double v = scratch[f];
  for (int b = 1; b < nb; b++) v += scratch[(long long)b * MAXF + f];
  out[f] = v;
}

bool device_ptr(const void* p) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

}  // namespace

extern "C" {

int hz_noalloc_setup(void) {
  double* p = nullptr;
  return noalloc_scratch(&p);
}

int hz_sum_fields_noalloc(const void* fields_dev, int nfields, long long ncell, int dtype, double* sums_dev,
                          void* cuda_stream) {
  if (!fields_dev || !sums_dev || nfields < 1 || ncell < 1 || (dtype != HZ_F32 && dtype != HZ_F64)) return HZ_EINVAL;
  // sizes beyond the fixed scratch (or beyond what one call is specified for) are refused, not truncated
  if (nfields > MAXF || ncell > HZ_NOALLOC_MAX_CELLS) return HZ_ELIMIT;
  if (!device_ptr(fields_dev) || !device_ptr(sums_dev)) return HZ_EINVAL;
  double* scratch = nullptr;
  const int rc = noalloc_scratch(&scratch);   // the device address, never the host-side name g_scratch
  if (rc) return rc;
  const long long want = (ncell + NT - 1) / NT;
  const int nb = (int)(want < MAXB ? want : MAXB);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  if (dtype == HZ_F64) k_sum_partials<double><<<nb, NT, 0, s>>>((const double*)fields_dev, nfields, ncell, scratch);
  else k_sum_partials<float><<<nb, NT, 0, s>>>((const float*)fields_dev, nfields, ncell, scratch);
  if (cudaGetLastError() != cudaSuccess) return HZ_ECUDA;
  k_sum_fold<<<1, 32, 0, s>>>(scratch, nb, nfields, sums_dev);
  if (cudaGetLastError() != cudaSuccess) return HZ_ECUDA;
  return HZ_OK;
}

}  // extern "C"
