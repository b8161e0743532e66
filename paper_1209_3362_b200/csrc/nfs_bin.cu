// nfs_bin.cu — step S6 of the hot path: averages over pairs and deterministic azimuthal binning
// ("azimuthally averaged power spectra"; readings R6-R10 in DESIGN.md).
//
// The |q|-bin of every half-plane Fourier pixel is precomputed on the host with exact integer
// arithmetic and the pixels are grouped by bin (perm / bin_start), each entry carrying its Hermitian
// weight (2 for 0 < kx < W/2, 1 for kx in {0, W/2}).  One CTA reduces one (row, bin) segment in a
// fixed order: per-thread strided fp64 sums, then a fixed shuffle/shared tree — no float atomics, so
// results are bit-identical from run to run.
#include "nfs_common.cuh"

namespace nfs {

// value of the static spectrum at pixel p: I2d = (sum|F'|^2 + 2 Re(sum F' conj F_r)) / N + |F_r|^2
__device__ __forceinline__ double i2d_value(const double* __restrict__ I2, const double2* __restrict__ I1,
                                            const float2* __restrict__ Fref, int64_t p, double invN) {
  const float2 fr = Fref[p];
  const double2 s1 = I1[p];
  const double rx = (double)fr.x, ry = (double)fr.y;
  return (I2[p] + 2.0 * (s1.x * rx + s1.y * ry)) * invN + (rx * rx + ry * ry);
}

// value of the variance-form spectrum at pixel p (half the plateau
// of Eq. 1): V2d = <|F_t - <F>_t|^2>_t = sum|F'|^2 / N - |sum F'|^2 / N^2.  The variance does not depend on the
// reference frame subtracted before the transform, so F_r does not enter; F' = F - F_0 is of the size of the
// fluctuations, so the difference does not cancel.
__device__ __forceinline__ double v2d_value(const double* __restrict__ I2, const double2* __restrict__ I1, int64_t p,
                                            double invN) {
  const double2 s1 = I1[p];
  const double mx = s1.x * invN, my = s1.y * invN;
  return fmax(I2[p] * invN - (mx * mx + my * my), 0.0);
}

// grid (n_qbins, n_lags + 2), 128 threads.  Row l < n_lags: D(b, tau_l); row n_lags: I(b); row n_lags + 1: V(b).
// binned != nullptr (bin-only mode): the D rows come from the weighted bin sums kept by k_bin_accumulate.
__global__ void __launch_bounds__(128) k_bin(const double* __restrict__ totals, const double* __restrict__ binned,
                                             const double* __restrict__ I2,
                                             const double2* __restrict__ I1, const float2* __restrict__ Fref,
                                             const uint32_t* __restrict__ perm, const int32_t* __restrict__ bin_start,
                                             const long long* __restrict__ npairs, int n_lags, int n_qbins, int64_t P,
                                             int64_t N, double* __restrict__ out) {
  const int b = blockIdx.x, row = blockIdx.y;
  const int beg = bin_start[b], end = bin_start[b + 1];
  double inv;
  if (row < n_lags) {
    const long long np = npairs[row];  // frame pairs accumulated at this lag (N - tau for a whole stack on one context)
    inv = np > 0 ? 1.0 / (double)np : 0.0;
  } else {
    inv = N > 0 ? 1.0 / (double)N : 0.0;  // N: frames in the I sums
  }
  double acc = 0.0, wsum = 0.0;
  for (int i = beg + (int)threadIdx.x; i < end; i += 128) {
    const uint32_t e = perm[i];
    const int64_t p = (int64_t)(e & 0x7fffffffu);
    const double wgt = (e >> 31) ? 2.0 : 1.0;
    double v;
    if (row < n_lags)
      v = binned ? 0.0 : totals[(int64_t)row * P + p] * inv;
    else if (row == n_lags)
      v = i2d_value(I2, I1, Fref, p, inv);
    else
      v = v2d_value(I2, I1, p, inv);
    acc += wgt * v;
    wsum += wgt;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    acc += __shfl_xor_sync(0xffffffffu, acc, o);
    wsum += __shfl_xor_sync(0xffffffffu, wsum, o);
  }
  __shared__ double sa[4], sw[4];
  if ((threadIdx.x & 31) == 0) {
    sa[threadIdx.x >> 5] = acc;
    sw[threadIdx.x >> 5] = wsum;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = (sa[0] + sa[1]) + (sa[2] + sa[3]);
    const double w = (sw[0] + sw[1]) + (sw[2] + sw[3]);
    if (binned && row < n_lags) a = binned[(int64_t)row * n_qbins + b] * inv;
    out[(int64_t)row * n_qbins + b] = (w > 0.0 && inv > 0.0) ? a / w : 0.0;
  }
}

// bin-only mode (the full 2-D spectra need not be stored): binned[l_first + row][b] += sum over the
// bin's pixels of weight * scratch[row][p], the per-pixel pair sums one lag group accumulated in one batch.  Same
// fixed order as k_bin, one writer per address, launches stream ordered: bit-identical from run to run.
__global__ void __launch_bounds__(128) k_bin_accumulate(const double* __restrict__ scratch, const uint32_t* __restrict__ perm,
                                                        const int32_t* __restrict__ bin_start, int n_qbins, int64_t P,
                                                        double* __restrict__ binned) {
  const int b = blockIdx.x, row = blockIdx.y;
  const int beg = bin_start[b], end = bin_start[b + 1];
  double acc = 0.0;
  for (int i = beg + (int)threadIdx.x; i < end; i += 128) {
    const uint32_t e = perm[i];
    const double v = scratch[(int64_t)row * P + (int64_t)(e & 0x7fffffffu)];
    acc += (e >> 31) ? 2.0 * v : v;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  __shared__ double sa[4];
  if ((threadIdx.x & 31) == 0) sa[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) binned[(int64_t)row * n_qbins + b] += (sa[0] + sa[1]) + (sa[2] + sa[3]);
}

__global__ void __launch_bounds__(256) k_I2d(const double* __restrict__ I2, const double2* __restrict__ I1,
                                             const float2* __restrict__ Fref, int64_t P, int64_t N,
                                             double* __restrict__ dst) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p < P) dst[p] = i2d_value(I2, I1, Fref, p, 1.0 / (double)N);
}

__global__ void __launch_bounds__(256) k_V2d(const double* __restrict__ I2, const double2* __restrict__ I1, int64_t P,
                                             int64_t N, double* __restrict__ dst) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p < P) dst[p] = v2d_value(I2, I1, p, 1.0 / (double)N);
}

__global__ void __launch_bounds__(256) k_D2d(const double* __restrict__ tot, int64_t P, double inv,
                                             double* __restrict__ dst) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p < P) dst[p] = tot[p] * inv;
}

// partial sums of one context in a form that adds up over contexts (time-chunk sharding): the I sums
// relative to this context's reference frame become absolute, S2 = sum |F_t|^2 and S1 = sum F_t over its n own frames
__global__ void __launch_bounds__(256) k_absolute_I(const double* __restrict__ I2, const double2* __restrict__ I1,
                                                    const float2* __restrict__ Fref, int64_t P, double n,
                                                    double* __restrict__ S2, double2* __restrict__ S1) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  const float2 fr = Fref[p];
  const double2 s1 = I1[p];
  const double rx = (double)fr.x, ry = (double)fr.y;
  S2[p] = I2[p] + 2.0 * (s1.x * rx + s1.y * ry) + n * (rx * rx + ry * ry);
  S1[p] = make_double2(s1.x + n * rx, s1.y + n * ry);
}

int launch_absolute_I(Ctx& c, double* d_S2, double2* d_S1) {
  k_absolute_I<<<(unsigned)((c.P + 255) / 256), 256, 0, c.stream>>>(c.I2, c.I1, c.Fref, c.P, (double)frames_in_I(c), d_S2, d_S1);
  NFS_CUDA(c, cudaGetLastError());
  return 1;
}

int launch_bin(Ctx& c) {
  dim3 grid((unsigned)c.n_qbins, (unsigned)(c.n_lags + 2));
  ProfScope ps(c, kKBin);
  std::vector<long long> np((size_t)c.n_lags);
  for (int l = 0; l < c.n_lags; ++l) np[(size_t)l] = (long long)pair_count(c, l);
  if (!NFS_CUDA(c, cudaMemcpyAsync(c.d_npairs, np.data(), sizeof(long long) * np.size(), cudaMemcpyHostToDevice, c.stream))) return 0;
  k_bin<<<grid, 128, 0, c.stream>>>(c.totals, c.bin_only ? c.totals_b : nullptr, c.I2, c.I1, c.Fref, c.perm, c.bin_start,
                                    c.d_npairs, c.n_lags, c.n_qbins, c.P, frames_in_I(c), c.d_out);
  NFS_CUDA(c, cudaGetLastError());
  return 1;
}

// ---- per-|q| fit of Eq. 1 (reading R19 in DESIGN.md) -----------------------
// D(b,tau) = A_b [1 - exp(-Gamma_b tau)] + C_b by unweighted least squares over the lags that have a frame pair:
// A = 2a T I_s (plateau), C = 2a B (noise floor), f = exp(-Gamma tau).  Variable projection: for a trial x = log Gamma
// the pair (A, C) is the linear least-squares solution; chi2(x) is scanned on 64 grid points of
// [log(1e-3 / tau_max), log(1e2 / tau_min)] and refined by 48 golden-section steps around the best one.  One warp per
// |q| bin, the lags spread over its lanes, fixed shuffle tree: deterministic.  Everything in fp64.
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
struct Eq1Lin {
  double A, C, chi2;
};
__device__ __forceinline__ Eq1Lin eq1_linear(double x, const double* __restrict__ Db, int n_qbins,
                                             const long long* __restrict__ npairs, const int32_t* __restrict__ lags, int n_lags,
                                             int lane) {
  const double G = exp(x);
  double n = 0.0, Sg = 0.0, Sgg = 0.0, Sd = 0.0, Sgd = 0.0;
  for (int l = lane; l < n_lags; l += 32) {
    if (npairs[l] > 0) {
      const double g = -expm1(-G * (double)lags[l]), d = Db[(int64_t)l * n_qbins];
      n += 1.0, Sg += g, Sgg += g * g, Sd += d, Sgd += g * d;
    }
  }
  n = warp_sum(n), Sg = warp_sum(Sg), Sgg = warp_sum(Sgg), Sd = warp_sum(Sd), Sgd = warp_sum(Sgd);
  Eq1Lin r;
  const double det = n * Sgg - Sg * Sg;
  if (det <= 1e-14 * n * Sgg) {
    r.A = 0.0;
    r.C = Sd / n;
  } else {
    r.A = (n * Sgd - Sg * Sd) / det;
    r.C = (Sd - r.A * Sg) / n;
  }
  double c2 = 0.0;
  for (int l = lane; l < n_lags; l += 32) {
    if (npairs[l] > 0) {
      const double g = -expm1(-G * (double)lags[l]);
      const double e = Db[(int64_t)l * n_qbins] - r.A * g - r.C;
      c2 += e * e;
    }
  }
  r.chi2 = warp_sum(c2);
  return r;
}

// grid: ceil(n_qbins / 4) CTAs of 4 warps.  D = binned structure function [n_lags][n_qbins]; fit = [4][n_qbins]: A, C, Gamma, chi2
__global__ void __launch_bounds__(128) k_fit_eq1(const double* __restrict__ D, const long long* __restrict__ npairs,
                                                 const int32_t* __restrict__ lags, const int32_t* __restrict__ bin_start,
                                                 int n_lags, int n_qbins, double* __restrict__ fit) {
  const int b = (int)blockIdx.x * 4 + ((int)threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (b >= n_qbins) return;
  int used = 0, tmin = 0x7fffffff, tmax = 0;
  for (int l = lane; l < n_lags; l += 32) {
    if (npairs[l] > 0) {
      ++used;
      tmin = min(tmin, lags[l]);
      tmax = max(tmax, lags[l]);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    used += __shfl_xor_sync(0xffffffffu, used, o);
    tmin = min(tmin, __shfl_xor_sync(0xffffffffu, tmin, o));
    tmax = max(tmax, __shfl_xor_sync(0xffffffffu, tmax, o));
  }
  double A = 0.0, C = 0.0, G = 0.0, chi2 = 0.0;
  if (used >= 3 && bin_start[b + 1] > bin_start[b]) {
    const double* Db = D + b;
    const double lo = log(1e-3 / (double)tmax), hi = log(1e2 / (double)tmin);
    constexpr int K = 64;
    int kbest = 0;
    double cbest = 0.0;
    for (int k = 0; k < K; ++k) {
      const double c2 = eq1_linear(lo + (hi - lo) * (double)k / (double)(K - 1), Db, n_qbins, npairs, lags, n_lags, lane).chi2;
      if (k == 0 || c2 < cbest) cbest = c2, kbest = k;
    }
    double a = lo + (hi - lo) * (double)max(kbest - 1, 0) / (double)(K - 1);
    double c = lo + (hi - lo) * (double)min(kbest + 1, K - 1) / (double)(K - 1);
    const double inv_phi = 0.61803398874989484820;
    double x1 = c - inv_phi * (c - a), x2 = a + inv_phi * (c - a);
    double f1 = eq1_linear(x1, Db, n_qbins, npairs, lags, n_lags, lane).chi2;
    double f2 = eq1_linear(x2, Db, n_qbins, npairs, lags, n_lags, lane).chi2;
    for (int it = 0; it < 48; ++it) {
      if (f1 <= f2) {
        c = x2, x2 = x1, f2 = f1;
        x1 = c - inv_phi * (c - a);
        f1 = eq1_linear(x1, Db, n_qbins, npairs, lags, n_lags, lane).chi2;
      } else {
        a = x1, x1 = x2, f1 = f2;
        x2 = a + inv_phi * (c - a);
        f2 = eq1_linear(x2, Db, n_qbins, npairs, lags, n_lags, lane).chi2;
      }
    }
    const double x = 0.5 * (a + c);
    const Eq1Lin r = eq1_linear(x, Db, n_qbins, npairs, lags, n_lags, lane);
    A = r.A, C = r.C, G = exp(x), chi2 = r.chi2;
  }
  if (lane == 0) {
    fit[b] = A;
    fit[(int64_t)n_qbins + b] = C;
    fit[2 * (int64_t)n_qbins + b] = G;
    fit[3 * (int64_t)n_qbins + b] = chi2;
  }
}

// after launch_bin (d_out and d_npairs are up to date): d_fit = [4][n_qbins]
int launch_fit_eq1(Ctx& c) {
  ProfScope ps(c, kKBin);
  k_fit_eq1<<<(unsigned)((c.n_qbins + 3) / 4), 128, 0, c.stream>>>(c.d_out, c.d_npairs, c.d_lags, c.bin_start, c.n_lags, c.n_qbins,
                                                                 c.d_fit);
  NFS_CUDA(c, cudaGetLastError());
  return 1;
}

int launch_bin_accumulate(Ctx& c, int l_first, int n_rows) {
  dim3 grid((unsigned)c.n_qbins, (unsigned)n_rows);
  ProfScope ps(c, kKBin);
  k_bin_accumulate<<<grid, 128, 0, c.stream>>>(c.totals, c.perm, c.bin_start, c.n_qbins, c.P,
                                               c.totals_b + (size_t)l_first * c.n_qbins);
  NFS_CUDA(c, cudaGetLastError());
  return 1;
}

int launch_I2d(Ctx& c, double* d_dst) {
  k_I2d<<<(unsigned)((c.P + 255) / 256), 256, 0, c.stream>>>(c.I2, c.I1, c.Fref, c.P, frames_in_I(c), d_dst);
  NFS_CUDA(c, cudaGetLastError());
  return 1;
}

int launch_V2d(Ctx& c, double* d_dst) {
  k_V2d<<<(unsigned)((c.P + 255) / 256), 256, 0, c.stream>>>(c.I2, c.I1, c.P, frames_in_I(c), d_dst);
  NFS_CUDA(c, cudaGetLastError());
  return 1;
}

int launch_D2d(Ctx& c, int l, double* d_dst) {
  const int64_t np = pair_count(c, l);
  const double inv = np > 0 ? 1.0 / (double)np : 0.0;
  k_D2d<<<(unsigned)((c.P + 255) / 256), 256, 0, c.stream>>>(c.totals + (int64_t)l * c.P, c.P, inv, d_dst);
  NFS_CUDA(c, cudaGetLastError());
  return 1;
}

}  // namespace nfs
