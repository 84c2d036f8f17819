// kh_divB_noalloc: the corner-centred divergence of kh_divB (S15a: the divergence Flux-CT preserves) for callers that
// cannot allocate -- code under CUDA-graph capture, serving loops, harnesses that forbid cudaMalloc.  include/kharm.h has the
// contract.  This file calls no cudaMalloc / cudaFree / allocating library routine: the reduction's scratch is the file-scope
// array below, which every GPU that loads libkharm.so holds until the process exits (KH_NOALLOC_SCRATCH_BYTES, ~0.5 MB).
//
// Two stages in ONE launch: every block leaves the maximum of its corners in scratch[32 + block]; the block that arrives last
// at the counter scratch[0] folds the partial maxima and writes the result.  The array is shared by every call and keeps the
// last call's contents: the counter is cleared (cudaMemsetAsync, no allocation) before each launch, the partials are all
// rewritten before they are read.  Calls that overlap on the GPU (two streams, two host threads) race on it.
#include <cuda_runtime.h>

#include <mutex>

#include "../../include/kharm.h"

namespace {

constexpr int NGH = 3;                 // ghost layers of the padded layout (KH_NGH)
constexpr int THREADS = 256;
constexpr int HEADER = 32;             // 256 B: the arrival counter sits alone in the first 256 B
constexpr long MAX_BLOCKS = KH_NOALLOC_MAX_CORNERS / THREADS;

static __device__ __align__(256) unsigned long long kh_noalloc_scratch[HEADER + MAX_BLOCKS];
static_assert(sizeof(kh_noalloc_scratch) == KH_NOALLOC_SCRATCH_BYTES, "kharm.h states the size of the static scratch");

// In host code `kh_noalloc_scratch` is a host-side stand-in, not a device address: the kernel gets the address that
// cudaGetSymbolAddress returns, looked up once per device with that device current.
constexpr int MAX_DEVICES = 64;
std::mutex g_lock;
unsigned long long* g_scratch[MAX_DEVICES] = {};

int scratch_of_current_device(unsigned long long** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) { cudaGetLastError(); return KH_ECUDA; }
  std::lock_guard<std::mutex> hold(g_lock);
  if (!g_scratch[dev]) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, kh_noalloc_scratch) != cudaSuccess || !p) { cudaGetLastError(); return KH_ECUDA; }
    g_scratch[dev] = static_cast<unsigned long long*>(p);
  }
  *out = g_scratch[dev];
  return KH_OK;
}

struct DivArgs {
  int n1, n2, n3;          // interior zones
  int lo1, lo2, lo3;       // first corner of each direction (0: the lower boundary plane is included)
  int c1, c2, c3;          // corners per direction
  double idx1, idx2, idx3; // 1 / dx
};

__device__ __forceinline__ long zone(const DivArgs& a, int i, int j, int k) {
  return ((long)(k + NGH) * (a.n2 + 2 * NGH) + (j + NGH)) * (a.n1 + 2 * NGH) + (i + NGH);
}
__device__ __forceinline__ long column(const DivArgs& a, int i, int j) { return (long)(j + NGH) * (a.n1 + 2 * NGH) + (i + NGH); }

// |div B| at corner (i - 1/2, j - 1/2, k - 1/2): for each direction d the difference of sqrt(-g) B^d across the corner,
// averaged over the four zone pairs that share it -- the same sums in the same order as kh_divB's kernel.
__device__ double corner_div(const DivArgs& a, const double* __restrict__ B, const double* __restrict__ gdet, int i, int j, int k) {
  const long nt = (long)(a.n1 + 2 * NGH) * (a.n2 + 2 * NGH) * (a.n3 + 2 * NGH);
  double div = 0.0;
  for (int d = 0; d < 3; d++) {
    double s = 0.0;
    for (int bb = 0; bb < 2; bb++)
      for (int aa = 0; aa < 2; aa++) {
        int o[3] = {0, 0, 0};
        o[(d + 1) % 3] = -aa; o[(d + 2) % 3] = -bb;
        const int ih = i + o[0], jh = j + o[1], kh = k + o[2];
        const int il = ih - (d == 0), jl = jh - (d == 1), kl = kh - (d == 2);
        const double gh = gdet ? gdet[column(a, ih, jh)] : 1.0, gl = gdet ? gdet[column(a, il, jl)] : 1.0;
        s += gh * B[d * nt + zone(a, ih, jh, kh)] - gl * B[d * nt + zone(a, il, jl, kl)];
      }
    div += 0.25 * s * (d == 0 ? a.idx1 : (d == 1 ? a.idx2 : a.idx3));
  }
  return fabs(div);
}

__global__ void __launch_bounds__(THREADS)
divb_noalloc_kernel(DivArgs a, const double* __restrict__ B, const double* __restrict__ gdet, unsigned long long* __restrict__ scratch,
                    double* __restrict__ max_abs) {
  __shared__ double part[THREADS / 32];
  __shared__ bool last;
  const long t = (long)blockIdx.x * THREADS + threadIdx.x, total = (long)a.c1 * a.c2 * a.c3;
  double m = 0.0;
  if (t < total) {
    const int i = (int)(t % a.c1) + a.lo1;
    const long r = t / a.c1;
    m = corner_div(a, B, gdet, i, (int)(r % a.c2) + a.lo2, (int)(r / a.c2) + a.lo3);
    if (!(m == m)) m = __longlong_as_double(0x7ff0000000000000LL);      // a NaN must not vanish in the fmax: report +inf
  }
  auto block_max = [&](double v) {
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = v;
    __syncthreads();
    double w = part[0];
    for (int q = 1; q < THREADS / 32; q++) w = fmax(w, part[q]);
    __syncthreads();
    return w;
  };
  m = block_max(m);
  if (threadIdx.x == 0) {
    scratch[HEADER + blockIdx.x] = (unsigned long long)__double_as_longlong(m);
    __threadfence();                                                    // the partial is visible before the arrival is
    last = atomicAdd(scratch, 1ULL) == (unsigned long long)gridDim.x - 1ULL;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  double w = 0.0;
  for (unsigned b = threadIdx.x; b < gridDim.x; b += THREADS)
    w = fmax(w, __longlong_as_double((long long)__ldcg(scratch + HEADER + b)));
  w = block_max(w);
  if (threadIdx.x == 0) {
    *max_abs = w;
    scratch[0] = 0ULL;                                                  // leave the counter as the next call needs it
  }
}

}  // namespace

extern "C" int kh_divB_noalloc(const double* B, const double* gdet, int n1, int n2, int n3, double dx1, double dx2, double dx3,
                               int lower_mask, double* max_abs, void* cuda_stream) {
  if (!B || !max_abs || n1 < 1 || n2 < 1 || n3 < 1 || !(dx1 > 0.0) || !(dx2 > 0.0) || !(dx3 > 0.0) || (lower_mask & ~7)) return KH_EINVAL;
  DivArgs a;
  a.n1 = n1; a.n2 = n2; a.n3 = n3;
  a.lo1 = (lower_mask & 1) ? 0 : 1; a.lo2 = (lower_mask & 2) ? 0 : 1; a.lo3 = (lower_mask & 4) ? 0 : 1;
  a.c1 = n1 - a.lo1; a.c2 = n2 - a.lo2; a.c3 = n3 - a.lo3;
  a.idx1 = 1.0 / dx1; a.idx2 = 1.0 / dx2; a.idx3 = 1.0 / dx3;
  const long long total = (long long)a.c1 * a.c2 * a.c3;
  if (total > KH_NOALLOC_MAX_CORNERS) return KH_ESIZE;                  // beyond the static scratch: nothing was enqueued
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  if (total == 0) return cudaMemsetAsync(max_abs, 0, sizeof(double), stream) == cudaSuccess ? KH_OK : (cudaGetLastError(), KH_ECUDA);
  unsigned long long* scratch = nullptr;
  if (int rc = scratch_of_current_device(&scratch)) return rc;
  if (cudaMemsetAsync(scratch, 0, HEADER * sizeof(unsigned long long), stream) != cudaSuccess) { cudaGetLastError(); return KH_ECUDA; }
  const unsigned blocks = (unsigned)((total + THREADS - 1) / THREADS);
  divb_noalloc_kernel<<<blocks, THREADS, 0, stream>>>(a, B, gdet, scratch, max_abs);
  if (cudaGetLastError() != cudaSuccess) return KH_ECUDA;
  return KH_OK;
}
