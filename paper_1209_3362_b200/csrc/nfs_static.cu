// nfs_static.cu — nfs_azimuthal_mean_static: the azimuthal average of step S6 ("azimuthally averaged
// power spectra"; readings R6, R7 in DESIGN.md) for callers that must not allocate device memory.
//
// Who that is.  The context-based path (nfs_create ... nfs_finalize) plans and cudaMallocs all of its buffers, the
// bin map among them, when a context is created.  Some programs cannot afford that call at the point where they need
// a |q| profile:
//   * an acquisition loop that analyses spectra at camera rate: cudaMalloc / cudaFree synchronise the whole device
//     and take an unpredictable time, so nothing on the per-frame path may allocate;
//   * a process whose device memory belongs, all of it, to somebody else's pool (a framework's caching allocator, a
//     fixed arena carved out at start-up, a MIG / MPS share with a hard limit): a cudaMalloc from inside a library
//     either fails there or takes memory behind the owner's back;
//   * plug-ins and callbacks that are only handed device pointers and a stream and are told not to touch the
//     allocator at all.
// For them this file offers one stand-alone call: device pointers in, device pointers out, no context, and the only
// working memory a fixed array that is part of the library image.
//
// How.  k_bin (nfs_bin.cu) walks a host-built, cudaMalloc'ed table of the pixels of every bin.  The variant here has no
// table: each pixel's bin is recomputed with exact integer arithmetic, every CTA reduces a fixed set of image rows into
// per-warp shared-memory bins in a fixed order, writes one partial sum and one weight per bin into the static scratch
// array, and a second kernel adds the CTAs' partials in CTA order.  No floating-point atomics anywhere: the result is
// bit-identical from run to run.
//
// The scratch array (kScratchDoubles doubles = 2.3 MiB) is a file-scope __device__ array: every GPU on which this
// library's module gets loaded holds its own copy until the process exits, used or not.  In HOST code its name is only
// a handle for the runtime, not a device address, so the address is asked for once per device with
// cudaGetSymbolAddress (device_state below) and that pointer is what the kernels receive.
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "../../include/nfs.h"

namespace {

constexpr int kMaxBins = NFS_STATIC_MAX_QBINS;  // largest n_qbins the scratch is sized for
constexpr int kMaxCtas = 148;                   // CTAs of the first kernel: one per SM of a B200, fewer for small frames
constexpr int kWarps = 4;                       // warps per CTA
constexpr int kThreads = 32 * kWarps;
constexpr size_t kScratchDoubles = (size_t)kMaxCtas * 2 * kMaxBins;  // per CTA: [n_qbins] weighted sums, [n_qbins] weights

static __device__ __align__(256) double g_static_scratch[kScratchDoubles];

// |q| bin of the Fourier pixel with |signed indices| (sx, sy) of an L x L frame: b = floor(n_b |q| / q_Nyquist), i.e.
// b^2 L^2 <= 4 n_b^2 (sx^2 + sy^2) < (b + 1)^2 L^2 (reading R6).  The square root only proposes b; the two integer
// comparisons decide it, so the result is exact.  -1: the DC pixel (R7) and everything at or beyond q_Nyquist.
// Largest intermediate: 4 * 1024^2 * 2 * 2048^2 = 2^45.
__device__ __forceinline__ int qbin_exact(int sx, int sy, int L, int nb) {
  const unsigned long long m = (unsigned long long)(sx * sx + sy * sy);
  if (m == 0ull) return -1;
  const unsigned long long L2 = (unsigned long long)L * (unsigned long long)L;
  const unsigned long long v = 4ull * (unsigned long long)nb * (unsigned long long)nb * m;
  if (v >= (unsigned long long)nb * (unsigned long long)nb * L2) return -1;
  long long b = (long long)(2.0 * (double)nb * sqrt((double)m) / (double)L);
  while (b > 0 && (unsigned long long)(b * b) * L2 > v) --b;
  while ((unsigned long long)((b + 1) * (b + 1)) * L2 <= v) ++b;
  return (int)b;
}

// grid G <= kMaxCtas CTAs of kThreads threads; dynamic shared memory kWarps * nb doubles + nb unsigned.
// spec = [L][L/2+1] (ky in FFT order, kx = 0..L/2).  CTA c takes the rows c, c + G, ...; warp w of it the pixels
// 32 w .. 32 w + 31, then + 128, ... of a row.  part[(2 c) nb + b] = sum of weight * value over the CTA's pixels of bin b,
// part[(2 c + 1) nb + b] = sum of the weights (Hermitian weight 2 for 0 < kx < L/2, else 1).  Every slot of the CTA is
// written, zeros included: the second kernel never reads anything an earlier call left behind.
__global__ void __launch_bounds__(kThreads) k_azimuthal_partial(const double* __restrict__ spec, int L, int nb,
                                                                double* __restrict__ part) {
  extern __shared__ double s_acc[];  // [kWarps][nb]
  unsigned* s_wgt = reinterpret_cast<unsigned*>(s_acc + (size_t)kWarps * nb);  // [nb], integer: order does not matter
  __shared__ double s_val[kWarps][32];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int n = L / 2;
  for (int i = tid; i < kWarps * nb; i += kThreads) s_acc[i] = 0.0;
  for (int i = tid; i < nb; i += kThreads) s_wgt[i] = 0u;
  __syncthreads();
  double* acc = s_acc + (size_t)warp * nb;
  for (int y = blockIdx.x; y < L; y += gridDim.x) {
    const int sy = y < L - y ? y : L - y;
    const double* row = spec + (size_t)y * (size_t)(n + 1);
    for (int x0 = 32 * warp; x0 <= n; x0 += kThreads) {  // trip count is the same for the whole warp
      const int x = x0 + lane;
      int b = -1;
      double wv = 0.0;
      if (x <= n) {
        b = qbin_exact(x, sy, L, nb);
        if (b >= 0) {
          const unsigned w = (x == 0 || x == n) ? 1u : 2u;
          wv = (double)w * row[x];
          atomicAdd(&s_wgt[b], w);
        }
      }
      // lanes that fell into the same bin: the lowest of them adds their values in lane order
      s_val[warp][lane] = wv;
      __syncwarp();
      const unsigned peers = __match_any_sync(0xffffffffu, b);
      if (b >= 0 && lane == __ffs(peers) - 1) {
        double a = 0.0;
        for (unsigned r = peers; r; r &= r - 1) a += s_val[warp][__ffs(r) - 1];
        acc[b] += a;
      }
      __syncwarp();
    }
  }
  __syncthreads();
  double* mine = part + (size_t)blockIdx.x * 2 * nb;
  for (int b = tid; b < nb; b += kThreads) {
    mine[b] = (s_acc[b] + s_acc[nb + b]) + (s_acc[2 * nb + b] + s_acc[3 * nb + b]);
    mine[nb + b] = (double)s_wgt[b];
  }
}

// one thread per bin: the partials of the G CTAs in CTA order; mean = sum / weight (empty bin: 0.0 / 0)
__global__ void __launch_bounds__(kThreads) k_azimuthal_reduce(const double* __restrict__ part, int G, int nb,
                                                               double* __restrict__ mean_q, long long* __restrict__ counts) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= nb) return;
  double s = 0.0, w = 0.0;
  for (int c = 0; c < G; ++c) {
    s += part[(size_t)c * 2 * nb + b];
    w += part[(size_t)c * 2 * nb + nb + b];
  }
  mean_q[b] = w > 0.0 ? s / w : 0.0;
  if (counts) counts[b] = (long long)w;  // exact: weights are small integers
}

// Per-device set-up, done by the first call that finds a device current: the scratch array's address ON THAT DEVICE
// and its SM count.  Guarded by a mutex so that two host threads may make their first call at once.
constexpr int kMaxDevices = 64;
struct DeviceState {
  double* scratch = nullptr;
  int n_sm = 0;
};
DeviceState g_dev[kMaxDevices];
std::mutex g_dev_mutex;

int device_state(DeviceState* out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return NFS_ERR_CUDA;
  std::lock_guard<std::mutex> lock(g_dev_mutex);
  DeviceState& d = g_dev[dev];
  if (!d.scratch) {
    double* p = nullptr;
    // the array's name is a host-side stand-in here; this is the only way host code learns where it lives on `dev`
    if (cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_static_scratch) != cudaSuccess || !p) return NFS_ERR_CUDA;
    int n_sm = 0;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n_sm < 1) return NFS_ERR_CUDA;
    d.n_sm = n_sm;
    d.scratch = p;
  }
  *out = d;
  return NFS_OK;
}

bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }

}  // namespace

extern "C" int nfs_azimuthal_mean_static(const double* d_spec2d, int W, int H, int n_qbins, double* d_mean_q, int64_t* d_counts,
                                         void* cuda_stream) {
  if (!d_spec2d || !d_mean_q || n_qbins < 1) return NFS_ERR_INVALID_ARG;
  if (!is_pow2(W) || !is_pow2(H) || W < 32 || H < 32 || W > 4096 || H > 4096) return NFS_ERR_INVALID_ARG;
  if (W != H) return NFS_ERR_UNSUPPORTED;
  if (n_qbins > kMaxBins) return NFS_ERR_TOO_LARGE;  // the scratch array cannot grow: refuse, never spill over
  if ((reinterpret_cast<uintptr_t>(d_spec2d) & 7u) || (reinterpret_cast<uintptr_t>(d_mean_q) & 7u) ||
      (reinterpret_cast<uintptr_t>(d_counts) & 7u))
    return NFS_ERR_INVALID_ARG;
  DeviceState dev;
  const int rc = device_state(&dev);
  if (rc != NFS_OK) return rc;
  cudaStream_t stream = reinterpret_cast<cudaStream_t>(cuda_stream);
  const int G = H < kMaxCtas ? H : (dev.n_sm < kMaxCtas ? dev.n_sm : kMaxCtas);
  const size_t smem = sizeof(double) * (size_t)kWarps * n_qbins + sizeof(unsigned) * (size_t)n_qbins;  // <= 36 KB
  k_azimuthal_partial<<<G, kThreads, smem, stream>>>(d_spec2d, W, n_qbins, dev.scratch);
  k_azimuthal_reduce<<<(n_qbins + kThreads - 1) / kThreads, kThreads, 0, stream>>>(dev.scratch, G, n_qbins, d_mean_q,
                                                                                  reinterpret_cast<long long*>(d_counts));
  return cudaGetLastError() == cudaSuccess ? NFS_OK : NFS_ERR_CUDA;
}
