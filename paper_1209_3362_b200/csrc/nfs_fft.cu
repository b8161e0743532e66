// nfs_fft.cu — steps S1-S3 of the hot path: exact frame sums, normalisation,
// hand-written 2-D real-to-complex FFT, written into the HBM ring.  No cuFFT anywhere.
//
//   S1  S_t = sum_x I_t(x) exactly (uint64); i_t = I_t * (W H / S_t)
//   S2  row pass: FFT along x of d_t = i_t - r, two image rows per complex FFT    L25, L31 (linearity)
//   S3  column pass: FFT along y of every kx column, unitary scale, ring slot     L31-33
// r is the first normalised frame (fp32); subtracting it before the transform keeps the large static
// beam out of the fp32 FFT.  Differences F_t - F_{t+tau} are unchanged.
//
// One persistent kernel per push batch (k_fft<L>, L = W = H).  Its CTAs pull work items from a global
// queue in a fixed order that software-pipelines the three stages through L2:
//      step s:  [sum items of frame s] [row items of frame s-1] [column items of frame s-1-kDc]
// An item waits (acquire-spin on a per-frame counter) only for items that precede it in the queue, so
// every claimed item is held by a running CTA and the smallest unfinished item can always finish: no
// deadlock, no co-residency requirement.  The row pass writes its result transposed ([kx][y]) into a
// small ring of `slots` intermediate frames that never leaves L2; the column pass therefore reads and
// writes contiguous 8*H-byte rows, and the Fourier frame layout in the HBM ring is [kx = 0..W/2][ky].
//
// FFT core: L = 32*M.  A team of M threads (M <= 32: part of one warp) holds 32 complex points per
// thread in registers: pass 1 = 32-point DFT in registers over the stride-M sequence, one exchange
// through padded shared memory (pitch 33, conflict free), pass 2 = M-point DFTs in registers.
// L > 1024: a 32-point register pass over L/32 threads, then 32 independent FFTs of length L/32 done the
// same way by 2 or 4 lanes each.  Twiddles between passes come from fp64-computed tables laid out so
// that consecutive lanes read consecutive entries.
#include "nfs_common.cuh"

namespace nfs {

// ------------------------------------------------------------------------------------------------
// complex helpers and register DFTs
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}

// cos(2 pi m / 32), sin(2 pi m / 32) as literals (folded after unrolling)
__device__ __forceinline__ constexpr float cos32(int m) {
  m &= 31;
  if (m > 16) m = 32 - m;
  const bool neg = m > 8;
  if (neg) m = 16 - m;
  float c = 0.f;
  switch (m) {
    case 0: c = 1.0f; break;
    case 1: c = 0.98078528040323044913f; break;
    case 2: c = 0.92387953251128675613f; break;
    case 3: c = 0.83146961230254523708f; break;
    case 4: c = 0.70710678118654752440f; break;
    case 5: c = 0.55557023301960222474f; break;
    case 6: c = 0.38268343236508977173f; break;
    case 7: c = 0.19509032201612826785f; break;
    default: c = 0.f; break;
  }
  return neg ? -c : c;
}
__device__ __forceinline__ constexpr float sin32(int m) { return cos32(m - 8); }

// d * exp(-2 pi i m / 32), m a compile-time constant after unrolling (0 <= m < 16)
__device__ __forceinline__ float2 mul_w32(float2 d, int m) {
  if (m == 0) return d;
  if (m == 8) return make_float2(d.y, -d.x);
  if (m == 4) {
    const float h = 0.70710678118654752440f;
    return make_float2((d.x + d.y) * h, (d.y - d.x) * h);
  }
  if (m == 12) {
    const float h = 0.70710678118654752440f;
    return make_float2((d.y - d.x) * h, -(d.x + d.y) * h);
  }
  const float c = cos32(m), s = -sin32(m);  // w = c + i s
  return make_float2(fmaf(d.x, c, -d.y * s), fmaf(d.x, s, d.y * c));
}

// N-point DFT (N = 2^k <= 32), decimation in frequency, in place on u[0], u[1], ... u[N-1];
// result in bit-reversed order.
template <int N>
__device__ __forceinline__ void dif(float2* u) {
  if constexpr (N >= 2) {
#pragma unroll
    for (int j = 0; j < N / 2; ++j) {
      const float2 a = u[j], b = u[j + N / 2];
      u[j] = cadd(a, b);
      u[j + N / 2] = mul_w32(csub(a, b), j * (32 / N));
    }
    dif<N / 2>(u);
    dif<N / 2>(u + N / 2);
  }
}
__host__ __device__ constexpr int bitrev(int k, int N) {
  int r = 0;
  for (int b = 1; b < N; b <<= 1) {
    r = (r << 1) | (k & 1);
    k >>= 1;
  }
  return r;
}
// natural order in, natural order out: X[k] = sum_t u[t] exp(-2 pi i t k / N)
template <int N>
__device__ __forceinline__ void dft(float2* u) {
  if constexpr (N >= 2) {
    dif<N>(u);
    float2 t[N];
#pragma unroll
    for (int k = 0; k < N; ++k) t[k] = u[bitrev(k, N)];
#pragma unroll
    for (int k = 0; k < N; ++k) u[k] = t[k];
  }
}

// ------------------------------------------------------------------------------------------------
// plan constants for FFT length L
// ------------------------------------------------------------------------------------------------
constexpr int kDr = 1;   // row items of frame f are queued kDr steps after its sum items
constexpr int kDc = 4;   // column items of frame f are queued kDc steps after its row items
constexpr int kSlots = 8;  // intermediate frames kept (all of them L2 resident)

template <int L>
struct Plan {
  static constexpr int T = L / 32;                       // threads per FFT
  static constexpr int NT = L <= 1024 ? 256 : 512;       // threads per CTA
  static constexpr int Fc = NT / T;                      // FFTs per CTA item
  static constexpr bool two = L > 1024;                  // two-level plan
  static constexpr int Mi = two ? L / 1024 : T;          // lanes per (inner) FFT
  static constexpr int Li = two ? L / 32 : L;            // inner FFT length
  static constexpr int pitchO = T + Mi;                  // two-level: pitch of the 32 inner sequences
  static constexpr int foot = two ? 32 * pitchO : T * 33;  // float2 per FFT buffer
  static constexpr int Sf = foot + ((2 - foot % 16) + 16) % 16;  // buffer stride == 2 (mod 16)
  static constexpr int n = L / 2;
  static constexpr int rowFfts = L / 2;                  // complex FFTs per frame in the row pass
  static constexpr int FcRow = Fc < rowFfts ? Fc : rowFfts;
  static constexpr int NR = (rowFfts + Fc - 1) / Fc;     // row items per frame
  static constexpr int NC = (n + 1 + Fc - 1) / Fc;       // column items per frame
  static constexpr int NS = L >= 256 ? 8 : 1;            // sum items per frame
  static constexpr int perStep = NS + NR + NC;
  static constexpr size_t smem = sizeof(float2) * ((size_t)Fc * Sf + 2 * Fc);
};

struct FftJob {
  const uint16_t* frames;     // [nf][H][W]  (mode 0)
  const float* ref;           // [H][W] fp32 reference r
  float2* rowT;               // [kSlots][(n+1)*H] row-pass output, transposed
  float2* dst;                // ring base (mode 0) or Fref (mode 1)
  unsigned long long* sums;   // [nf] exact frame sums
  unsigned int* cnt;          // [1 + 3 nf]: queue head, sum_done[nf], row_done[nf], col_done[nf]
  const float2* tw_in;        // [Li]  tw_in[j2*32 + k1] = exp(-2 pi i j2 k1 / Li)
  const float2* tw_out;       // [L]   tw_out[k1*T + j2] = exp(-2 pi i j2 k1 / L)   (two-level only)
  int* flags;
  long long t_first;
  int R;
  int nf;
  int mode;                   // 0: frames -> ring;  1: the reference itself -> Fref
  float scale;                // 1/sqrt(W H)
};

// ------------------------------------------------------------------------------------------------
// team FFT.  In: u[t] = x[t*T + tau].  Out: u[r] = X[out_index<L>(tau, r)].
// `buf` is this FFT's shared-memory buffer (Plan<L>::foot float2).  The caller guarantees that every
// thread of the team has finished reading `buf` before the call.
// ------------------------------------------------------------------------------------------------
template <int T>
__device__ __forceinline__ void team_sync(int team) {
  if constexpr (T <= 32) {
    __syncwarp();
  } else {
    asm volatile("bar.sync %0, %1;" ::"r"(team + 1), "r"(T) : "memory");
  }
}

// one level: L' = 32*M, M <= 32 lanes (all inside one warp).  buf: M*33 float2.
template <int M>
__device__ __forceinline__ void fft_level(float2 (&u)[32], float2* buf, int lam, const float2* __restrict__ tw) {
  dft<32>(u);
  if constexpr (M > 1) {
#pragma unroll
    for (int k1 = 0; k1 < 32; ++k1) buf[lam * 33 + k1] = u[k1];
    __syncwarp();
#pragma unroll
    for (int it = 0; it < 32 / M; ++it) {
      const int k1 = lam + M * it;
#pragma unroll
      for (int j2 = 0; j2 < M; ++j2) {
        float2 v = buf[j2 * 33 + k1];
        if (j2 > 0) v = cmul(v, __ldg(&tw[j2 * 32 + k1]));
        u[it * M + j2] = v;
      }
      dft<M>(&u[it * M]);
    }
  }
}

template <int L>
__device__ __forceinline__ void fft_team(float2 (&u)[32], float2* buf, int tau, int team, const FftJob& j) {
  using P = Plan<L>;
  if constexpr (!P::two) {
    fft_level<P::T>(u, buf, tau, j.tw_in);
  } else {
    dft<32>(u);  // over t -> k1; this thread is j2 = tau
#pragma unroll
    for (int k1 = 0; k1 < 32; ++k1) {
      float2 v = u[k1];
      if (k1 > 0) v = cmul(v, __ldg(&j.tw_out[k1 * P::T + tau]));
      buf[k1 * P::pitchO + tau] = v;
    }
    team_sync<P::T>(team);
    const int k1 = tau / P::Mi, lam = tau % P::Mi;
    float2* sb = buf + k1 * P::pitchO;
#pragma unroll
    for (int t = 0; t < 32; ++t) u[t] = sb[t * P::Mi + lam];
    __syncwarp();
    fft_level<P::Mi>(u, sb, lam, j.tw_in);
  }
}

// index k of the output held in register r of thread tau
template <int L>
__device__ __forceinline__ int out_index(int tau, int r) {
  using P = Plan<L>;
  if constexpr (!P::two) {
    return (tau + P::T * (r / P::T)) + 32 * (r % P::T);
  } else {
    const int k1 = tau / P::Mi, lam = tau % P::Mi;
    const int kk = (lam + P::Mi * (r / P::Mi)) + 32 * (r % P::Mi);
    return k1 + 32 * kk;
  }
}

// ------------------------------------------------------------------------------------------------
// queue helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned ld_acquire(const unsigned* p) {
  unsigned v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
// all threads call; returns when *p >= target (thread 0 spins)
__device__ __forceinline__ void wait_count(const unsigned* p, unsigned target) {
  if (threadIdx.x == 0) {
    while (ld_acquire(p) < target) __nanosleep(64);
  }
  __syncthreads();
}
// all threads call after their global writes
__device__ __forceinline__ void signal_count(unsigned* p) {
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(p, 1u);
  }
}

// scale 1/m_t = W H / S_t as an unevaluated fp32 pair (hi + lo), from fp64
__device__ __forceinline__ void frame_scale(unsigned long long S, float wh, float& hi, float& lo, int* flags) {
  if (S == 0ull) {
    hi = lo = 0.f;
    if (threadIdx.x == 0) atomicOr(flags, 1);
    return;
  }
  double s = (double)wh / (double)S;
  hi = (float)s;
  lo = (float)(s - (double)hi);
}

__device__ __forceinline__ void unpack8(uint4 v, float* p) {
  p[0] = (float)(v.x & 0xffffu); p[1] = (float)(v.x >> 16);
  p[2] = (float)(v.y & 0xffffu); p[3] = (float)(v.y >> 16);
  p[4] = (float)(v.z & 0xffffu); p[5] = (float)(v.z >> 16);
  p[6] = (float)(v.w & 0xffffu); p[7] = (float)(v.w >> 16);
}

// staging layout of the row pass: complex index j -> float2 slot, XOR swizzle on 16-byte units so
// that both the 128-bit staging stores and the stride-T pass-1 loads are bank-conflict free
__device__ __forceinline__ int stage_slot(int j) {
  const int a = j >> 1;
  return ((a ^ ((a >> 3) & 3)) << 1) | (j & 1);
}

// ------------------------------------------------------------------------------------------------
// items
// ------------------------------------------------------------------------------------------------
template <int L>
__device__ __forceinline__ void item_sum(const FftJob& j, int f, int part) {
  using P = Plan<L>;
  __shared__ unsigned long long s_part[P::NT / 32];
  if (j.mode == 0) {
    const int64_t n16 = (int64_t)L * L / 8;  // uint4 per frame
    const int64_t per = n16 / P::NS;
    const uint4* src = reinterpret_cast<const uint4*>(j.frames) + (int64_t)f * n16 + (int64_t)part * per;
    unsigned long long acc = 0;
    for (int64_t i0 = 0; i0 < per; i0 += (int64_t)P::NT * 4) {
      unsigned a32 = 0;  // <= 4 * 8 * 65535 < 2^32
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int64_t i = i0 + (int64_t)q * P::NT + threadIdx.x;
        if (i < per) {
          const uint4 v = __ldg(&src[i]);
          a32 += (v.x & 0xffffu) + (v.x >> 16) + (v.y & 0xffffu) + (v.y >> 16) + (v.z & 0xffffu) + (v.z >> 16) +
                 (v.w & 0xffffu) + (v.w >> 16);
        }
      }
      acc += a32;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
      unsigned long long t = 0;
      for (int w = 0; w < P::NT / 32; ++w) t += s_part[w];
      atomicAdd(&j.sums[f], t);  // integer: order independent, deterministic
    }
  }
  signal_count(&j.cnt[1 + f]);
}

template <int L>
__device__ __forceinline__ void item_row(const FftJob& j, int f, int blk, float2* sm) {
  using P = Plan<L>;
  constexpr int W = L, H = L, n = P::n;
  const int tid = threadIdx.x;
  const int team = tid / P::T, tau = tid % P::T;
  float2* nyq = sm + (size_t)P::Fc * P::Sf;  // [2 Fc]
  float2* buf = sm + (size_t)team * P::Sf;
  const unsigned nf = (unsigned)j.nf;

  // dependencies: this frame's sum; the column pass of the frame that used this slot before
  wait_count(&j.cnt[1 + f], (unsigned)P::NS);
  if (f >= kSlots) wait_count(&j.cnt[1 + 2 * nf + (f - kSlots)], (unsigned)P::NC);

  float hi = 0.f, lo = 0.f;
  if (j.mode == 0) frame_scale(__ldcg(&j.sums[f]), (float)W * (float)H, hi, lo, j.flags);

  int q = blk * P::Fc + team;         // complex FFT index: image rows 2q, 2q+1
  const bool valid = q < P::rowFfts;
  if (!valid) q = P::rowFfts - 1;
  const int64_t ra = (int64_t)(2 * q) * W, rb = ra + W;
  const uint16_t* fr = j.frames + (int64_t)f * W * H;

  // load + convert + normalise + subtract reference; stage z[j] = d_a[j] + i d_b[j]
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    const int c = tau + P::T * r;  // chunk of 8 pixels
    const float4 a0 = __ldg(reinterpret_cast<const float4*>(j.ref + ra + c * 8));
    const float4 a1 = __ldg(reinterpret_cast<const float4*>(j.ref + ra + c * 8 + 4));
    const float4 b0 = __ldg(reinterpret_cast<const float4*>(j.ref + rb + c * 8));
    const float4 b1 = __ldg(reinterpret_cast<const float4*>(j.ref + rb + c * 8 + 4));
    float da[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
    float db[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
    if (j.mode == 0) {
      float pa[8], pb[8];
      unpack8(__ldg(reinterpret_cast<const uint4*>(fr + ra + c * 8)), pa);
      unpack8(__ldg(reinterpret_cast<const uint4*>(fr + rb + c * 8)), pb);
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        da[i] = fmaf(pa[i], lo, fmaf(pa[i], hi, -da[i]));  // exact product, one rounding at |d|
        db[i] = fmaf(pb[i], lo, fmaf(pb[i], hi, -db[i]));
      }
    }
#pragma unroll
    for (int qq = 0; qq < 4; ++qq) {
      const int a = 4 * c + qq;
      const int as = a ^ ((a >> 3) & 3);
      reinterpret_cast<float4*>(buf)[as] = make_float4(da[2 * qq], db[2 * qq], da[2 * qq + 1], db[2 * qq + 1]);
    }
  }
  team_sync<P::T>(team);
  float2 u[32];
#pragma unroll
  for (int t = 0; t < 32; ++t) u[t] = buf[stage_slot(t * P::T + tau)];
  team_sync<P::T>(team);
  fft_team<L>(u, buf, tau, team, j);
  team_sync<P::T>(team);
#pragma unroll
  for (int r = 0; r < 32; ++r) buf[out_index<L>(tau, r)] = u[r];
  team_sync<P::T>(team);

  // untangle the two real rows: A[k] = (Z[k] + conj Z[L-k]) / 2,  B[k] = (Z[k] - conj Z[L-k]) / (2i).
  // In place: slot k <- A[k], slot L-k <- B[k] (1 <= k < n); slot 0 <- A[0], slot n <- B[0]; Nyquist aside.
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    const int k = tau + P::T * i;
    if (k == 0) {
      const float2 z0 = buf[0], zh = buf[n];
      buf[0] = make_float2(z0.x, 0.f);
      buf[n] = make_float2(z0.y, 0.f);
      nyq[2 * team] = make_float2(zh.x, 0.f);
      nyq[2 * team + 1] = make_float2(zh.y, 0.f);
    } else {
      const float2 zk = buf[k], zm = buf[L - k];
      buf[k] = make_float2(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y));
      buf[L - k] = make_float2(0.5f * (zk.y + zm.y), -0.5f * (zk.x - zm.x));
    }
  }
  __syncthreads();

  // transposed store: rowT[slot][kx][y], 16 bytes (rows 2q, 2q+1) per thread and kx
  float2* out = j.rowT + (size_t)(f % kSlots) * ((size_t)(n + 1) * H);
  const int y0 = blk * P::Fc * 2;
  constexpr int FcR = P::FcRow;
  for (int e = tid; e < n * FcR; e += P::NT) {
    const int kxl = e & 1, ft = (e >> 1) % FcR, kx = 2 * (e / (2 * FcR)) + kxl;
    const float2* b = sm + (size_t)ft * P::Sf;
    const float2 A = b[kx], B = b[kx ? L - kx : n];
    *reinterpret_cast<float4*>(out + (size_t)kx * H + y0 + 2 * ft) = make_float4(A.x, A.y, B.x, B.y);
  }
  if (tid < FcR) {
    *reinterpret_cast<float4*>(out + (size_t)n * H + y0 + 2 * tid) =
        make_float4(nyq[2 * tid].x, nyq[2 * tid].y, nyq[2 * tid + 1].x, nyq[2 * tid + 1].y);
  }
  signal_count(&j.cnt[1 + nf + f]);
}

template <int L>
__device__ __forceinline__ void item_col(const FftJob& j, int f, int blk, float2* sm) {
  using P = Plan<L>;
  constexpr int H = L, n = P::n;
  const int tid = threadIdx.x;
  const int team = tid / P::T, tau = tid % P::T;
  float2* buf = sm + (size_t)team * P::Sf;
  const unsigned nf = (unsigned)j.nf;

  wait_count(&j.cnt[1 + nf + f], (unsigned)P::NR);

  int q = blk * P::Fc + team;  // kx row
  const bool valid = q <= n;
  if (!valid) q = n;
  const float2* src = j.rowT + (size_t)(f % kSlots) * ((size_t)(n + 1) * H) + (size_t)q * H;
  float2 u[32];
#pragma unroll
  for (int t = 0; t < 32; ++t) u[t] = __ldcg(&src[t * P::T + tau]);
  fft_team<L>(u, buf, tau, team, j);
  if (valid) {
    const int64_t Pn = (int64_t)(n + 1) * H;
    const int slot = (j.R > 0) ? (int)((j.t_first + f) % j.R) : 0;
    float2* dst = j.dst + (int64_t)slot * Pn + (int64_t)q * H;
    const float sc = j.scale;
#pragma unroll
    for (int r = 0; r < 32; ++r) dst[out_index<L>(tau, r)] = make_float2(u[r].x * sc, u[r].y * sc);
  }
  signal_count(&j.cnt[1 + 2 * nf + f]);
}

// ------------------------------------------------------------------------------------------------
// the persistent kernel
// ------------------------------------------------------------------------------------------------
template <int L>
__global__ void __launch_bounds__(Plan<L>::NT, (L <= 1024 ? 2 : 1)) k_fft(const FftJob j) {
  using P = Plan<L>;
  extern __shared__ __align__(16) float2 sm[];
  __shared__ unsigned s_item;
  const unsigned total = (unsigned)(j.nf + kDr + kDc) * P::perStep;
  unsigned nxt = 0;
  if (threadIdx.x == 0) nxt = atomicAdd(&j.cnt[0], 1u);
  for (;;) {
    if (threadIdx.x == 0) s_item = nxt;
    __syncthreads();
    const unsigned item = s_item;
    if (item >= total) break;
    if (threadIdx.x == 0) nxt = atomicAdd(&j.cnt[0], 1u);  // prefetch the next claim
    const int s = (int)(item / P::perStep), r = (int)(item % P::perStep);
    if (r < P::NS) {
      if (s < j.nf) {
        item_sum<L>(j, s, r);
        continue;
      }
    } else if (r < P::NS + P::NR) {
      const int f = s - kDr;
      if (f >= 0 && f < j.nf) {
        item_row<L>(j, f, r - P::NS, sm);
        continue;
      }
    } else {
      const int f = s - kDr - kDc;
      if (f >= 0 && f < j.nf) {
        item_col<L>(j, f, r - P::NS - P::NR, sm);
        continue;
      }
    }
    __syncthreads();  // no-op item: keep s_item's reader/writer ordering
  }
}

// ------------------------------------------------------------------------------------------------
// first frame only: exact sum and the reference image r(x) = fp32(I_0(x) / m_0)
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_frame_sum(const uint4* __restrict__ frame, int64_t n16,
                                                   unsigned long long* __restrict__ sum) {
  unsigned long long acc = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (int64_t)gridDim.x * blockDim.x) {
    const uint4 v = __ldg(&frame[i]);
    acc += (v.x & 0xffffu) + (v.x >> 16) + (v.y & 0xffffu) + (v.y >> 16) + (v.z & 0xffffu) + (v.z >> 16) +
           (v.w & 0xffffu) + (v.w >> 16);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  __shared__ unsigned long long part[8];
  if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long t = 0;
    for (int w = 0; w < 8; ++w) t += part[w];
    atomicAdd(sum, t);
  }
}

__global__ void __launch_bounds__(256) k_make_ref(const uint16_t* __restrict__ frame0, int64_t npx, float wh,
                                                  const unsigned long long* __restrict__ sums, float* __restrict__ ref,
                                                  int* flags) {
  float hi, lo;
  frame_scale(sums[0], wh, hi, lo, flags);
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < npx; i += (int64_t)gridDim.x * blockDim.x) {
    float v = (float)frame0[i];
    ref[i] = fmaf(v, lo, v * hi);
  }
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
template <int L>
static int launch_fft_L(Ctx& c, const FftJob& job, int cls) {
  using P = Plan<L>;
  if (c.fft_grid == 0) {
    cudaFuncSetAttribute(k_fft<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P::smem);
    int per_sm = 0, dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_fft<L>, P::NT, P::smem);
    if (per_sm < 1) per_sm = 1;
    c.fft_grid = per_sm * sms;
  }
  const long long total = (long long)(job.nf + kDr + kDc) * P::perStep;
  const int grid = (int)std::min<long long>(c.fft_grid, total);
  ProfScope ps(c, cls);
  cudaMemsetAsync(c.fft_cnt, 0, sizeof(unsigned) * (1 + 3 * (size_t)job.nf) + 0, c.stream);
  cudaMemsetAsync(c.sums, 0, sizeof(unsigned long long) * (size_t)job.nf, c.stream);
  k_fft<L><<<grid, P::NT, P::smem, c.stream>>>(job);
  return 1;
}

static int launch_fft(Ctx& c, const FftJob& job, int cls) {
  switch (c.W) {
    case 32: return launch_fft_L<32>(c, job, cls);
    case 64: return launch_fft_L<64>(c, job, cls);
    case 128: return launch_fft_L<128>(c, job, cls);
    case 256: return launch_fft_L<256>(c, job, cls);
    case 512: return launch_fft_L<512>(c, job, cls);
    case 1024: return launch_fft_L<1024>(c, job, cls);
    case 2048: return launch_fft_L<2048>(c, job, cls);
    case 4096: return launch_fft_L<4096>(c, job, cls);
    default: return 0;
  }
}

size_t fft_rowT_elems(const Ctx& c) { return (size_t)kSlots * (size_t)c.P; }

static FftJob make_job(Ctx& c) {
  FftJob j;
  j.frames = nullptr;
  j.ref = c.ref;
  j.rowT = c.rowbuf;
  j.dst = c.ring;
  j.sums = c.sums;
  j.cnt = c.fft_cnt;
  j.tw_in = c.tw;
  j.tw_out = c.tw_out;
  j.flags = c.d_flags;
  j.t_first = 0;
  j.R = c.R;
  j.nf = 0;
  j.mode = 0;
  j.scale = (float)(1.0 / sqrt((double)c.W * (double)c.H));
  return j;
}

// first pushed frame: S_0, r = fp32(I_0 / m_0), Fref = FFT(r)
int launch_make_ref(Ctx& c, const uint16_t* frame0) {
  const int64_t npx = (int64_t)c.W * c.H;
  {
    ProfScope ps(c, kKSum);
    cudaMemsetAsync(c.sums, 0, sizeof(unsigned long long), c.stream);
    int nblk = (int)std::min<int64_t>(592, (npx / 8 + 255) / 256);
    k_frame_sum<<<nblk, 256, 0, c.stream>>>(reinterpret_cast<const uint4*>(frame0), npx / 8, c.sums);
    nblk = (int)std::min<int64_t>(1184, (npx + 1023) / 1024);
    k_make_ref<<<nblk, 256, 0, c.stream>>>(frame0, npx, (float)c.W * (float)c.H, c.sums, c.ref, c.d_flags);
  }
  FftJob j = make_job(c);
  j.dst = c.Fref;
  j.R = 0;
  j.nf = 1;
  j.mode = 1;
  return 2 + launch_fft(c, j, kKFft);
}

// ring[t_first .. t_first + nf) = unitary FFT(i_t - r)
int launch_fft_frames(Ctx& c, const uint16_t* frames, int nf, int64_t t_first) {
  FftJob j = make_job(c);
  j.frames = frames;
  j.nf = nf;
  j.t_first = t_first;
  return launch_fft(c, j, kKFft);
}

}  // namespace nfs
