// nfs_fft.cu — steps S1-S3 of the hot path: exact frame sums, normalisation,
// hand-written 2-D real-to-complex FFT (row pass + column pass), written into the HBM ring.
//
//   S1  S_t = sum_x I_t(x) exactly (uint64); i_t = I_t * (W H / S_t)
//   S2  row pass: W-point real->complex FFT of every row of d_t = i_t - r     L25, L31 (linearity)
//   S3  column pass: H-point complex FFT of every column, unitary scale        L31-33
// r is the first normalised frame (fp32); subtracting it before the transform keeps the large
// static beam out of the fp32 FFT.  Differences F_t - F_{t+tau} are unchanged.
// The FFT is a shared-memory Stockham autosort, radix 8 with a final radix 2/4 pass, twiddles
// from an fp64-computed table.  No cuFFT anywhere.
#include "nfs_common.cuh"

namespace nfs {

// ------------------------------------------------------------------------------------------------
// complex helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ float2 cmul_mi(float2 a) { return make_float2(a.y, -a.x); }  // a * (-i)
__device__ __forceinline__ void bfly2(float2& a, float2& b) {
  float2 t = a;
  a = cadd(t, b);
  b = csub(t, b);
}

// R-point DFT in registers; input natural order, output natural order (X[k] = sum_t u[t] w_R^{tk}).
template <int R>
__device__ __forceinline__ void dft(float2* u);
template <>
__device__ __forceinline__ void dft<1>(float2*) {}
template <>
__device__ __forceinline__ void dft<2>(float2* u) { bfly2(u[0], u[1]); }
template <>
__device__ __forceinline__ void dft<4>(float2* u) {
  bfly2(u[0], u[2]);
  bfly2(u[1], u[3]);
  u[3] = cmul_mi(u[3]);
  bfly2(u[0], u[1]);
  bfly2(u[2], u[3]);
  // now u0=X0, u1=X2, u2=X1, u3=X3
  float2 t = u[1];
  u[1] = u[2];
  u[2] = t;
}
template <>
__device__ __forceinline__ void dft<8>(float2* u) {
  const float h = 0.70710678118654752440f;
  bfly2(u[0], u[4]);
  bfly2(u[1], u[5]);
  bfly2(u[2], u[6]);
  bfly2(u[3], u[7]);
  u[5] = make_float2((u[5].x + u[5].y) * h, (u[5].y - u[5].x) * h);   // * w8^1
  u[6] = cmul_mi(u[6]);                                               // * w8^2
  u[7] = make_float2((u[7].y - u[7].x) * h, -(u[7].x + u[7].y) * h);  // * w8^3
  // two radix-4 on (0,1,2,3) and (4,5,6,7), outputs bit-reversed
  bfly2(u[0], u[2]);
  bfly2(u[1], u[3]);
  u[3] = cmul_mi(u[3]);
  bfly2(u[0], u[1]);
  bfly2(u[2], u[3]);
  bfly2(u[4], u[6]);
  bfly2(u[5], u[7]);
  u[7] = cmul_mi(u[7]);
  bfly2(u[4], u[5]);
  bfly2(u[6], u[7]);
  // u0=X0 u1=X4 u2=X2 u3=X6 u4=X1 u5=X5 u6=X3 u7=X7  -> natural order
  float2 x1 = u[4], x2 = u[2], x3 = u[6], x4 = u[1], x5 = u[5], x6 = u[3];
  u[1] = x1;
  u[2] = x2;
  u[3] = x3;
  u[4] = x4;
  u[5] = x5;
  u[6] = x6;
}

// One Stockham pass of radix R over a length-len FFT held in shared memory with element stride
// `es` (1 for rows, Cw for column tiles).  `g` in [0, len/8) is this thread's butterfly slot; every
// thread owns exactly 8 elements per pass (8/R butterflies).  p = product of the radices done so far.
// Twiddle table tw[j] = exp(-2 pi i j / twN), twN a multiple of len.
// Caller: load_pass -> __syncthreads -> store_pass -> __syncthreads.
template <int R>
__device__ __forceinline__ void pass_load(const float2* s, int es, int len, int g, float2* u) {
  constexpr int IPT = 8 / R;
  const int T = len / R, g8 = len >> 3;
#pragma unroll
  for (int it = 0; it < IPT; ++it) {
    const int i = g + it * g8;
#pragma unroll
    for (int t = 0; t < R; ++t) u[it * R + t] = s[(i + t * T) * es];
  }
}
template <int R>
__device__ __forceinline__ void pass_store(float2* s, int es, int len, int g, int p, float2* u,
                                           const float2* __restrict__ tw, int twN) {
  constexpr int IPT = 8 / R;
  const int g8 = len >> 3;
  const int tstep = twN / (p * R);  // table index of exp(-2 pi i / (p R))
#pragma unroll
  for (int it = 0; it < IPT; ++it) {
    const int i = g + it * g8;
    const int k = i & (p - 1);
    const int j = (i - k) * R + k;
    float2* v = u + it * R;
    if (p > 1) {
#pragma unroll
      for (int t = 1; t < R; ++t) v[t] = cmul(v[t], __ldg(&tw[t * k * tstep]));
    }
    dft<R>(v);
#pragma unroll
    for (int t = 0; t < R; ++t) s[(j + t * p) * es] = v[t];
  }
}

// Full length-len FFT (len = 8^a * {1,2,4}, len >= 16) of the sequence s[g*es], in place.
// All threads of the CTA must call it (it contains __syncthreads); `active` masks idle threads.
__device__ __forceinline__ void fft_smem(float2* s, int es, int len, int g, bool active, const float2* __restrict__ tw,
                                         int twN) {
  float2 u[8];
  int p = 1, rem = len;
  while (rem >= 8) {
    if (active) pass_load<8>(s, es, len, g, u);
    __syncthreads();
    if (active) pass_store<8>(s, es, len, g, p, u, tw, twN);
    __syncthreads();
    p <<= 3;
    rem >>= 3;
  }
  if (rem == 4) {
    if (active) pass_load<4>(s, es, len, g, u);
    __syncthreads();
    if (active) pass_store<4>(s, es, len, g, p, u, tw, twN);
    __syncthreads();
  } else if (rem == 2) {
    if (active) pass_load<2>(s, es, len, g, u);
    __syncthreads();
    if (active) pass_store<2>(s, es, len, g, p, u, tw, twN);
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------------
// S1: exact integer frame sums (reading R3).  grid (nblk, nf), 256 threads.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_frame_sum(const uint4* __restrict__ frames, int64_t n16_per_frame,
                                                   unsigned long long* __restrict__ sums) {
  const uint4* f = frames + (int64_t)blockIdx.y * n16_per_frame;
  unsigned int acc = 0;  // <= 128 iterations * 8 * 65535 < 2^32 for every supported size
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16_per_frame;
       i += (int64_t)gridDim.x * blockDim.x) {
    uint4 v = __ldg(&f[i]);
    acc += (v.x & 0xffffu) + (v.x >> 16) + (v.y & 0xffffu) + (v.y >> 16) + (v.z & 0xffffu) + (v.z >> 16) +
           (v.w & 0xffffu) + (v.w >> 16);
  }
  unsigned long long a = acc;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
  __shared__ unsigned long long part[8];
  if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = a;
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long t = 0;
    for (int w = 0; w < 8; ++w) t += part[w];
    atomicAdd(&sums[blockIdx.y], t);  // integer: order independent, deterministic
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

// r(x) = fp32( I_0(x) / m_0 ): the reference image.  Any fixed image would do; only its exact fp32
// value matters, and every later frame and Fref use this same array.
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
// S2: row pass.  grid (H / rpc, nf); block = rpc * n/8 threads; dynamic smem = rpc*(n + 1) float2.
// MODE 0: input uint16 frame, d = I*s - r.   MODE 1: input is the fp32 reference itself.
// Output rowbuf[f] in Fourier-frame layout: main [H][n] + Nyquist [H].
// ------------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(1024) k_row(const uint16_t* __restrict__ frames, const float* __restrict__ ref,
                                               const unsigned long long* __restrict__ sums, float2* __restrict__ rowbuf,
                                               const float2* __restrict__ tw, int W, int H, int rpc, int* flags) {
  extern __shared__ float2 sm[];
  const int n = W >> 1, tpr = n >> 3;
  const int tid = threadIdx.x, nthr = blockDim.x;
  const int f = blockIdx.y, y0 = blockIdx.x * rpc;
  float2* nyq = sm + rpc * n;
  float hi = 0.f, lo = 0.f;
  if (MODE == 0) frame_scale(sums[f], (float)W * (float)H, hi, lo, flags);

  // load + convert + subtract reference: 8 pixels (4 packed complex points) per item
  const int items = rpc * (n >> 2);
  for (int e = tid; e < items; e += nthr) {
    const int row = e / (n >> 2), c4 = e - row * (n >> 2);
    const int64_t off = (int64_t)(y0 + row) * W + c4 * 8;
    const float4 r0 = __ldg(reinterpret_cast<const float4*>(ref + off));
    const float4 r1 = __ldg(reinterpret_cast<const float4*>(ref + off + 4));
    float d[8];
    if (MODE == 0) {
      const uint4 v = __ldg(reinterpret_cast<const uint4*>(frames + (int64_t)f * W * H + off));
      const float p[8] = {(float)(v.x & 0xffffu), (float)(v.x >> 16), (float)(v.y & 0xffffu), (float)(v.y >> 16),
                          (float)(v.z & 0xffffu), (float)(v.z >> 16), (float)(v.w & 0xffffu), (float)(v.w >> 16)};
      const float rr[8] = {r0.x, r0.y, r0.z, r0.w, r1.x, r1.y, r1.z, r1.w};
#pragma unroll
      for (int q = 0; q < 8; ++q) d[q] = fmaf(p[q], lo, fmaf(p[q], hi, -rr[q]));  // exact product, one rounding at |d|
    } else {
      d[0] = r0.x; d[1] = r0.y; d[2] = r0.z; d[3] = r0.w;
      d[4] = r1.x; d[5] = r1.y; d[6] = r1.z; d[7] = r1.w;
    }
    float4* dst = reinterpret_cast<float4*>(sm + row * n + c4 * 4);
    dst[0] = make_float4(d[0], d[1], d[2], d[3]);
    dst[1] = make_float4(d[4], d[5], d[6], d[7]);
  }
  __syncthreads();

  // n-point complex FFT of z[j] = x[2j] + i x[2j+1], one row per tpr threads
  const int row = tid / tpr, g = tid - row * tpr;
  // tw has W entries exp(-2 pi i j / W); the n-point FFT needs exp(-2 pi i /(p R)) = tw[W/(p R)]: twN = W.
  fft_smem(sm + row * n, 1, n, g, true, tw, W);

  // real-to-complex post-processing: X[k] = E + w O, X[n-k] = conj(E - w O), w = exp(-2 pi i k / W)
  const int half = n >> 1;
  for (int e = tid; e < rpc * half; e += nthr) {
    const int r = e / half, k = e - r * half;
    float2* z = sm + r * n;
    if (k == 0) {
      const float2 z0 = z[0], zh = z[half];
      z[0] = make_float2(z0.x + z0.y, 0.f);
      nyq[r] = make_float2(z0.x - z0.y, 0.f);
      z[half] = make_float2(zh.x, -zh.y);
    } else {
      const float2 a = z[k], b = z[n - k];
      const float2 E = make_float2(0.5f * (a.x + b.x), 0.5f * (a.y - b.y));
      const float2 O = make_float2(0.5f * (a.y + b.y), 0.5f * (b.x - a.x));
      const float2 wO = cmul(__ldg(&tw[k]), O);
      z[k] = cadd(E, wO);
      const float2 m = csub(E, wO);
      z[n - k] = make_float2(m.x, -m.y);
    }
  }
  __syncthreads();

  // store: main rows as float4 (2 complex), Nyquist column
  float2* out = rowbuf + (int64_t)f * ((int64_t)H * (n + 1));
  for (int e = tid; e < rpc * half; e += nthr) {
    const int r = e / half, c2 = e - r * half;
    reinterpret_cast<float4*>(out + (int64_t)(y0 + r) * n)[c2] = reinterpret_cast<const float4*>(sm + r * n)[c2];
  }
  if (tid < rpc) out[(int64_t)H * n + y0 + tid] = nyq[tid];
}

// ------------------------------------------------------------------------------------------------
// S3: column pass.  grid (n/Cw + 1, nf): tiles of Cw main-block columns, last block = Nyquist column.
// smem = H*Cw float2.  Writes scale * FFT_y into dst frame (ring slot (t_first+f) mod R, or Fref).
// ------------------------------------------------------------------------------------------------
template <int LF>
__global__ void __launch_bounds__(1024) k_col(const float2* __restrict__ rowbuf, float2* __restrict__ dst_base,
                                               int64_t t_first, int R, const float2* __restrict__ tw, int W, int H,
                                               int Cw, float scale) {
  extern __shared__ float2 sm[];
  const int n = W >> 1;
  const int tid = threadIdx.x, nthr = blockDim.x;
  const int f = blockIdx.y;
  const int64_t P = (int64_t)H * (n + 1);
  const bool is_nyq = (blockIdx.x == (unsigned)(n / Cw));
  const int ncols = is_nyq ? 1 : Cw;
  const int64_t base = is_nyq ? (int64_t)H * n : (int64_t)blockIdx.x * Cw;
  const int pitch = is_nyq ? 1 : n;
  const float2* src = rowbuf + (int64_t)f * P + base;
  const int slot = (R > 0) ? (int)((t_first + f) % R) : 0;
  float2* dst = dst_base + (int64_t)slot * P + base;

  for (int e = tid; e < H * Cw; e += nthr) {
    const int y = e / Cw, c = e - y * Cw;
    if (c < ncols) sm[e] = src[(int64_t)y * pitch + c];
  }
  __syncthreads();

  // every thread owns LF butterfly slots b = tid + lf*nthr in [0, (H/8)*Cw); column c = b % Cw
  {
    float2 u[LF][8];
    int p = 1, rem = H;
    auto run = [&](auto Rtag) {
      constexpr int RR = decltype(Rtag)::value;
#pragma unroll
      for (int lf = 0; lf < LF; ++lf) {
        const int b = tid + lf * nthr, c = b % Cw, g = b / Cw;
        if (c < ncols) pass_load<RR>(sm + c, Cw, H, g, u[lf]);
      }
      __syncthreads();
#pragma unroll
      for (int lf = 0; lf < LF; ++lf) {
        const int b = tid + lf * nthr, c = b % Cw, g = b / Cw;
        if (c < ncols) pass_store<RR>(sm + c, Cw, H, g, p, u[lf], tw, H);
      }
      __syncthreads();
    };
    while (rem >= 8) {
      run(std::integral_constant<int, 8>{});
      p <<= 3;
      rem >>= 3;
    }
    if (rem == 4) run(std::integral_constant<int, 4>{});
    if (rem == 2) run(std::integral_constant<int, 2>{});
  }

  for (int e = tid; e < H * Cw; e += nthr) {
    const int y = e / Cw, c = e - y * Cw;
    if (c < ncols) {
      float2 v = sm[e];
      dst[(int64_t)y * pitch + c] = make_float2(v.x * scale, v.y * scale);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
static int col_cw(int H) { return H > 2048 ? 4 : 8; }

int launch_frame_sums(Ctx& c, const uint16_t* frames, int nf) {
  const int64_t n16 = (int64_t)c.W * c.H / 8;
  int nblk = (int)((n16 + 256 * 8 - 1) / (256 * 8));
  if (nblk > 64) nblk = 64;
  if (nblk < 1) nblk = 1;
  ProfScope ps(c, kKSum);
  cudaMemsetAsync(c.sums, 0, sizeof(unsigned long long) * nf, c.stream);
  k_frame_sum<<<dim3(nblk, nf), 256, 0, c.stream>>>(reinterpret_cast<const uint4*>(frames), n16, c.sums);
  return 1;
}

int launch_make_ref(Ctx& c, const uint16_t* frame0) {
  const int64_t npx = (int64_t)c.W * c.H;
  int nblk = (int)((npx + 1023) / 1024);
  if (nblk > 1184) nblk = 1184;
  ProfScope ps(c, kKSum);
  k_make_ref<<<nblk, 256, 0, c.stream>>>(frame0, npx, (float)c.W * (float)c.H, c.sums, c.ref, c.d_flags);
  return 1;
}

static void row_cfg(const Ctx& c, int& rpc, int& threads, size_t& smem) {
  const int tpr = c.n / 8;
  rpc = 256 / tpr;
  if (rpc < 1) rpc = 1;
  if (rpc > c.H) rpc = c.H;
  threads = rpc * tpr;
  smem = sizeof(float2) * (size_t)rpc * (c.n + 1);
}

template <int MODE>
static int launch_row(Ctx& c, const uint16_t* frames, int nf) {
  int rpc, threads;
  size_t smem;
  row_cfg(c, rpc, threads, smem);
  ProfScope ps(c, kKRow);
  k_row<MODE><<<dim3(c.H / rpc, nf), threads, smem, c.stream>>>(frames, c.ref, c.sums, c.rowbuf, c.tw, c.W, c.H, rpc,
                                                              c.d_flags);
  return 1;
}

static int launch_col(Ctx& c, float2* dst, int64_t t_first, int R, int nf) {
  const int Cw = col_cw(c.H);
  const int slots = (c.H / 8) * Cw;
  const int threads = slots > 1024 ? 1024 : slots;
  const int lf = slots / threads;
  const size_t smem = sizeof(float2) * (size_t)c.H * Cw;
  const float scale = (float)(1.0 / sqrt((double)c.W * (double)c.H));
  dim3 grid(c.n / Cw + 1, nf);
  ProfScope ps(c, kKCol);
  if (lf == 1) {
    if (smem > 48 * 1024) cudaFuncSetAttribute(k_col<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    k_col<1><<<grid, threads, smem, c.stream>>>(c.rowbuf, dst, t_first, R, c.tw, c.W, c.H, Cw, scale);
  } else {
    if (smem > 48 * 1024) cudaFuncSetAttribute(k_col<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    k_col<2><<<grid, threads, smem, c.stream>>>(c.rowbuf, dst, t_first, R, c.tw, c.W, c.H, Cw, scale);
  }
  return 1;
}

int launch_fft_ref(Ctx& c) {
  int n = launch_row<1>(c, nullptr, 1);
  n += launch_col(c, c.Fref, 0, 0, 1);
  return n;
}

int launch_fft_frames(Ctx& c, const uint16_t* frames, int nf, int64_t t_first) {
  int n = launch_row<0>(c, frames, nf);
  n += launch_col(c, c.ring, t_first, c.R, nf);
  return n;
}

}  // namespace nfs
