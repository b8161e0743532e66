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
//      step s:  [sum items of frame s] [row items of frame s-Dr] [column items of frame s-Dr-Dc]
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
#include <algorithm>

#include "nfs_common.cuh"

namespace nfs {

// ------------------------------------------------------------------------------------------------
// complex helpers and register DFTs
// ------------------------------------------------------------------------------------------------
// complex add / subtract as one packed instruction (SASS FADD2): one issue slot instead of two
__device__ __forceinline__ float2 cadd(float2 a, float2 b) {
  unsigned long long ua, ub, ur;
  asm("mov.b64 %0, {%1, %2};" : "=l"(ua) : "f"(a.x), "f"(a.y));
  asm("mov.b64 %0, {%1, %2};" : "=l"(ub) : "f"(b.x), "f"(b.y));
  asm("add.f32x2 %0, %1, %2;" : "=l"(ur) : "l"(ua), "l"(ub));
  float2 r;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(ur));
  return r;
}
__device__ __forceinline__ float2 csub(float2 a, float2 b) {
  unsigned long long ua, ub, ur;
  asm("mov.b64 %0, {%1, %2};" : "=l"(ua) : "f"(a.x), "f"(a.y));
  asm("mov.b64 %0, {%1, %2};" : "=l"(ub) : "f"(b.x), "f"(b.y));
  asm("sub.f32x2 %0, %1, %2;" : "=l"(ur) : "l"(ua), "l"(ub));
  float2 r;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(ur));
  return r;
}
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
// L2 eviction hints: the uint16 frame is read by the sum items and again, a few queue
// steps later, by the row items; the row-pass intermediate is written and re-read through L2; the ring
// slot is written once and not read again by this kernel.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long pol_evict_last() {
  unsigned long long p;
  asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ unsigned long long pol_evict_first() {
  unsigned long long p;
  asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ uint4 ld_u4_hint(const uint4* p, unsigned long long pol) {
  uint4 v;
  asm volatile("ld.global.nc.L2::cache_hint.v4.u32 {%0, %1, %2, %3}, [%4], %5;"
               : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
               : "l"(p), "l"(pol));
  return v;
}
__device__ __forceinline__ float2 ld_f2_cg_hint(const float2* p, unsigned long long pol) {
  float2 v;
  asm volatile("ld.global.cg.L2::cache_hint.v2.f32 {%0, %1}, [%2], %3;" : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(pol) : "memory");
  return v;
}
__device__ __forceinline__ void st_f2_hint(float2* p, float2 v, unsigned long long pol) {
  asm volatile("st.global.L2::cache_hint.v2.f32 [%0], {%1, %2}, %3;" ::"l"(p), "f"(v.x), "f"(v.y), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_f4_hint(float4* p, float4 v, unsigned long long pol) {
  asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w),
               "l"(pol)
               : "memory");
}

// ------------------------------------------------------------------------------------------------
// plan constants for FFT length L
// ------------------------------------------------------------------------------------------------
constexpr int kMaxSlots = 40;

template <int L>
struct Plan {
  static constexpr int T = L / 32;                       // threads per FFT
  static constexpr int NT = (L == 512 || L == 1024) ? 128 : 256;  // threads per CTA
  static constexpr int minBlocks = L == 1024 ? 5 : 512 / NT;  // CTAs per SM the kernel is compiled for (1024: 96 registers, no spill)
  static constexpr int Fc = NT / T;                      // FFTs per CTA item
  static constexpr bool two = L > 1024;                  // two-level plan
  static constexpr int Mi = two ? L / 1024 : T;          // lanes per (inner) FFT
  static constexpr int Li = two ? L / 32 : L;            // inner FFT length
  static constexpr int pitchO = T + Mi;                  // two-level: pitch of the 32 inner sequences
  static constexpr int foot = two ? 32 * pitchO : T * 33;  // float2 per FFT buffer
  // buffer stride == 16 / (FFTs per item) (mod 16) float2: the transposed store reads element kx of every FFT of the
  // item side by side, one 8-byte bank each within a half-warp
  // (even, so that every buffer stays 16-byte aligned for the 128-bit staging stores)
  static constexpr int padTo = Fc >= 8 ? 2 : (Fc >= 4 ? 4 : 8);
  static constexpr int Sf = foot + ((padTo - foot % 16) + 16) % 16;
  static constexpr int n = L / 2;
  static constexpr int rowFfts = L / 2;                  // complex FFTs per frame in the row pass
  static constexpr int FcRow = Fc < rowFfts ? Fc : rowFfts;
  static constexpr int NR = (rowFfts + Fc - 1) / Fc;     // row items per frame
  static constexpr int NC = (n + 1 + Fc - 1) / Fc;       // column items per frame
  static constexpr int NS = L >= 256 ? 8 * 256 / NT : 1;  // sum items per frame
  static constexpr int perStep = NS + NR + NC;
  static constexpr size_t smem = sizeof(float2) * ((size_t)Fc * Sf + 2 * Fc);
  // Queue distances, in steps (one step = the items of one frame).  About 2 * (resident CTAs) items are
  // claimed at any time (each CTA holds the item it runs and the next one), i.e. `win` steps; an item
  // should find its dependencies finished, so they are queued more than `win` steps earlier.
  // The write-after-read dependency on an intermediate slot needs Dc < slots (it must precede in the queue).
  static constexpr int claimed = 2 * minBlocks * 148;
  static constexpr int win_ = (claimed + perStep - 1) / perStep;
  static constexpr int win = win_ < 16 ? win_ : 16;
  static constexpr int Dr = win + 1;                   // sum items -> row items
  static constexpr int Dc = L <= 1024 ? win + 1 : win;  // row items -> column items
  static constexpr int slots = Dc + win + (L <= 1024 ? 1 : 0);  // intermediate frames
  static_assert(Dc < slots && slots <= kMaxSlots, "queue order must cover the slot reuse dependency");
};

struct FftJob {
  const uint16_t* frames;     // [nf][H][W]  (mode 0)
  const float* ref;           // [H][W] fp32 reference r
  float2* rowT;               // [slots][(n+1)*H] row-pass output, transposed
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
// queue helpers.  Completion counters only ever grow, so a value read early (prefetched while the
// previous item was running) that already satisfies the target stays valid.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned ld_relaxed(const unsigned* p) {
  unsigned v;
  asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
// thread 0 only: spin until *p >= target, starting from the prefetched value `seen`
__device__ __forceinline__ void spin_until(const unsigned* p, unsigned target, unsigned seen) {
  while (seen < target) {
    __nanosleep(32);
    seen = ld_relaxed(p);
  }
}
// acquire side: orders this thread's later loads after the counter loads above; the CTA barrier that
// follows extends that order to the other threads.  Data produced by other CTAs is then read with
// __ldcg (L2), never through a possibly stale L1 line.
__device__ __forceinline__ void acquire_fence() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
// all threads call after their global writes (release side)
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

// uint16 -> fp32 without the conversion unit (I2F runs at a quarter of the FP32 rate): 2^23 + v is exact in fp32 for
// v < 2^23, so OR-ing v into the mantissa of 2^23 and subtracting 2^23 gives float(v) with one logic op and one add
__device__ __forceinline__ float u16f(unsigned v) { return __uint_as_float(0x4b000000u | v) - 8388608.0f; }
__device__ __forceinline__ void unpack8(uint4 v, float* p) {
  p[0] = u16f(v.x & 0xffffu); p[1] = u16f(v.x >> 16);
  p[2] = u16f(v.y & 0xffffu); p[3] = u16f(v.y >> 16);
  p[4] = u16f(v.z & 0xffffu); p[5] = u16f(v.z >> 16);
  p[6] = u16f(v.w & 0xffffu); p[7] = u16f(v.w >> 16);
}

// staging layout of the row pass: complex index j -> float2 slot, XOR swizzle on 16-byte units so
// that both the 128-bit staging stores and the stride-T pass-1 loads are bank-conflict free
__device__ __forceinline__ int stage_slot(int j) {
  const int a = j >> 1;
  return ((a ^ ((a >> 3) & 3)) << 1) | (j & 1);
}

// a decoded work item and its dependencies (all on items that precede it in the queue)
struct Item {
  int type;  // 0 sum, 1 row, 2 column, 3 nothing to do
  int f;     // frame within the batch
  int blk;   // part / row block / column block
};
template <int L>
__device__ __forceinline__ Item decode_item(unsigned item, int nf) {
  using P = Plan<L>;
  Item it;
  const int s = (int)(item / P::perStep), r = (int)(item % P::perStep);
  if (r < P::NS) {
    it.type = 0, it.f = s, it.blk = r;
  } else if (r < P::NS + P::NR) {
    it.type = 1, it.f = s - P::Dr, it.blk = r - P::NS;
  } else {
    it.type = 2, it.f = s - P::Dr - P::Dc, it.blk = r - P::NS - P::NR;
  }
  if (it.f < 0 || it.f >= nf) it.type = 3;
  return it;
}
// first dependency: row <- sum_done[f] == NS; column <- row_done[f] == NR
template <int L>
__device__ __forceinline__ const unsigned* dep_a(const FftJob& j, const Item& it, unsigned& target) {
  using P = Plan<L>;
  if (it.type == 1) {
    target = (unsigned)P::NS;
    return &j.cnt[1 + it.f];
  }
  if (it.type == 2) {
    target = (unsigned)P::NR;
    return &j.cnt[1 + j.nf + it.f];
  }
  target = 0;
  return nullptr;
}
// second dependency (write-after-read on the intermediate slot): row(f) <- col_done[f - slots] == NC
template <int L>
__device__ __forceinline__ const unsigned* dep_b(const FftJob& j, const Item& it, unsigned& target) {
  using P = Plan<L>;
  if (it.type == 1 && it.f >= P::slots) {
    target = (unsigned)P::NC;
    return &j.cnt[1 + 2 * j.nf + (it.f - P::slots)];
  }
  target = 0;
  return nullptr;
}

// ------------------------------------------------------------------------------------------------
// items
// ------------------------------------------------------------------------------------------------
template <int L>
__device__ __forceinline__ void item_sum(const FftJob& j, int f, int part, unsigned long long* s_part) {
  using P = Plan<L>;
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
          const uint4 v = ld_u4_hint(&src[i], pol_evict_last());
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

// one chunk of 8 pixels of image rows a and b, and of the reference
struct Chunk {
  float4 a0, a1, b0, b1;
  uint4 pa, pb;
};
__device__ __forceinline__ void chunk_load(Chunk& ck, const FftJob& j, const uint16_t* fr, int64_t ra, int64_t rb, int c) {
  ck.a0 = __ldg(reinterpret_cast<const float4*>(j.ref + ra + c * 8));
  ck.a1 = __ldg(reinterpret_cast<const float4*>(j.ref + ra + c * 8 + 4));
  ck.b0 = __ldg(reinterpret_cast<const float4*>(j.ref + rb + c * 8));
  ck.b1 = __ldg(reinterpret_cast<const float4*>(j.ref + rb + c * 8 + 4));
  if (j.mode == 0) {
    ck.pa = ld_u4_hint(reinterpret_cast<const uint4*>(fr + ra + c * 8), pol_evict_first());
    ck.pb = ld_u4_hint(reinterpret_cast<const uint4*>(fr + rb + c * 8), pol_evict_first());
  }
}
// convert + normalise + subtract the reference, stage z[j] = d_a[j] + i d_b[j]
__device__ __forceinline__ void chunk_stage(const Chunk& ck, int mode, float hi, float lo, float2* buf, int c) {
  float da[8] = {ck.a0.x, ck.a0.y, ck.a0.z, ck.a0.w, ck.a1.x, ck.a1.y, ck.a1.z, ck.a1.w};
  float db[8] = {ck.b0.x, ck.b0.y, ck.b0.z, ck.b0.w, ck.b1.x, ck.b1.y, ck.b1.z, ck.b1.w};
  if (mode == 0) {
    float pa[8], pb[8];
    unpack8(ck.pa, pa);
    unpack8(ck.pb, pb);
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

// ------------------------------------------------------------------------------------------------
// the persistent kernel
// ------------------------------------------------------------------------------------------------
template <int L>
__global__ void __launch_bounds__(Plan<L>::NT, Plan<L>::minBlocks) k_fft(const FftJob j) {
  using P = Plan<L>;
  constexpr int W = L, H = L, n = P::n;
  extern __shared__ __align__(16) float2 sm[];
  __shared__ unsigned s_item[2];
  __shared__ unsigned long long s_sum;
  __shared__ unsigned long long s_part[P::NT / 32];
  const int tid = threadIdx.x;
  const int team = tid / P::T, tau = tid % P::T;
  float2* buf = sm + (size_t)team * P::Sf;
  const unsigned total = (unsigned)(j.nf + P::Dr + P::Dc) * P::perStep;
  const size_t Pn = (size_t)(n + 1) * H;

  // thread 0 runs the queue two claims ahead: q1 = the next item, whose dependency counters it reads
  // while the current item is being processed (seenA / seenB)
  unsigned q1 = 0, seenA = 0, seenB = 0;
  if (tid == 0) {
    s_item[0] = atomicAdd(&j.cnt[0], 1u);
    q1 = atomicAdd(&j.cnt[0], 1u);
  }
  __syncthreads();

  for (int iter = 0;; ++iter) {
    const unsigned item = s_item[iter & 1];
    if (item >= total) break;
    const Item it = decode_item<L>(item, j.nf);
    unsigned tgtA, tgtB;
    const unsigned* pA = dep_a<L>(j, it, tgtA);
    const unsigned* pB = dep_b<L>(j, it, tgtB);
    unsigned curA = seenA, curB = seenB;  // prefetched for this item during the previous one
    if (tid == 0) {
      s_item[(iter + 1) & 1] = q1;
      unsigned tA, tB;
      const Item nx = q1 < total ? decode_item<L>(q1, j.nf) : Item{3, 0, 0};
      const unsigned* nA = dep_a<L>(j, nx, tA);
      const unsigned* nB = dep_b<L>(j, nx, tB);
      seenA = nA ? ld_relaxed(nA) : 0u;
      seenB = nB ? ld_relaxed(nB) : 0u;
      q1 = atomicAdd(&j.cnt[0], 1u);
      if (iter == 0) {  // nothing was prefetched for the very first item
        curA = pA ? ld_relaxed(pA) : 0u;
        curB = pB ? ld_relaxed(pB) : 0u;
      }
    }

    if (it.type == 0) {
      item_sum<L>(j, it.f, it.blk, s_part);
      continue;
    }
    if (it.type == 3) {
      __syncthreads();  // keeps the s_item double buffer ordered
      continue;
    }

    // ---------------- row or column item: load phase ----------------
    const int f = it.f;
    const bool is_row = it.type == 1;
    float2 u[32];
    int q = it.blk * P::Fc + team;  // row item: complex FFT index (image rows 2q, 2q+1); column item: kx
    bool valid;
    float2* rowT = j.rowT + (size_t)(f % P::slots) * Pn;
    if (is_row) {
      valid = q < P::rowFfts;
      if (!valid) q = P::rowFfts - 1;
      const int64_t ra = (int64_t)(2 * q) * W, rb = ra + W;
      const uint16_t* fr = j.frames + (int64_t)f * W * H;
      Chunk ck[2];
      chunk_load(ck[0], j, fr, ra, rb, tau);  // in flight while thread 0 checks this frame's sum
      if (tid == 0) {
        spin_until(pA, tgtA, curA);
        acquire_fence();
        s_sum = __ldcg(&j.sums[f]);
      }
      __syncthreads();
      float hi = 0.f, lo = 0.f;
      if (j.mode == 0) frame_scale(s_sum, (float)W * (float)H, hi, lo, j.flags);
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        if (r < 3) chunk_load(ck[(r + 1) & 1], j, fr, ra, rb, tau + P::T * (r + 1));
        chunk_stage(ck[r & 1], j.mode, hi, lo, buf, tau + P::T * r);
      }
      team_sync<P::T>(team);
#pragma unroll
      for (int t = 0; t < 32; ++t) u[t] = buf[stage_slot(t * P::T + tau)];
      team_sync<P::T>(team);
    } else {
      valid = q <= n;
      if (!valid) q = n;
      if (tid == 0) {
        spin_until(pA, tgtA, curA);
        acquire_fence();
      }
      __syncthreads();
      const float2* src = rowT + (size_t)q * H;
#pragma unroll
      for (int t = 0; t < 32; ++t) u[t] = ld_f2_cg_hint(&src[t * P::T + tau], pol_evict_first());
    }

    // ---------------- the FFT itself (one call site: the code is large) ----------------
    fft_team<L>(u, buf, tau, team, j);

    if (is_row) {
      team_sync<P::T>(team);
#pragma unroll
      for (int r = 0; r < 32; ++r) buf[out_index<L>(tau, r)] = u[r];
      team_sync<P::T>(team);
      // (the two real rows are untangled on the way out, below: no further pass over shared memory)
      // the intermediate slot must have been drained by the column pass of frame f - slots
      if (tid == 0 && pB) {
        spin_until(pB, tgtB, curB);
        acquire_fence();
      }
      __syncthreads();
      // transposed store: rowT[kx][y], 16 bytes (rows 2q, 2q+1) per thread and kx
      const int y0 = it.blk * P::Fc * 2;
      constexpr int FcR = P::FcRow;
      for (int e = tid; e < n * FcR; e += P::NT) {
        const int kxl = e & 1, ft = (e >> 1) % FcR, kx = 2 * (e / (2 * FcR)) + kxl;
        // untangle the two real rows packed into one complex FFT: A[k] = (Z[k] + conj Z[L-k]) / 2,
        // B[k] = (Z[k] - conj Z[L-k]) / (2i);  k = 0: A = Re Z[0], B = Im Z[0]
        const float2* b = sm + (size_t)ft * P::Sf;
        const float2 zk = b[kx], zm = b[kx ? L - kx : 0];
        const float4 v = kx ? make_float4(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y), 0.5f * (zk.y + zm.y), -0.5f * (zk.x - zm.x))
                            : make_float4(zk.x, 0.f, zk.y, 0.f);
        st_f4_hint(reinterpret_cast<float4*>(rowT + (size_t)kx * H + y0 + 2 * ft), v, pol_evict_last());
      }
      if (tid < FcR) {  // the Nyquist column: A = Re Z[n], B = Im Z[n]
        const float2 zh = sm[(size_t)tid * P::Sf + n];
        *reinterpret_cast<float4*>(rowT + (size_t)n * H + y0 + 2 * tid) = make_float4(zh.x, 0.f, zh.y, 0.f);
      }
      signal_count(&j.cnt[1 + j.nf + f]);
    } else {
      if (valid) {
        const int slot = (j.R > 0) ? (int)((j.t_first + f) % j.R) : 0;
        float2* dst = j.dst + (size_t)slot * Pn + (size_t)q * H;
        const float sc = j.scale;
#pragma unroll
        for (int r = 0; r < 32; ++r) st_f2_hint(&dst[out_index<L>(tau, r)], make_float2(u[r].x * sc, u[r].y * sc), pol_evict_first());
      }
      signal_count(&j.cnt[1 + 2 * j.nf + f]);
    }
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
static bool configure_L(Ctx& c) {
  using P = Plan<L>;
  if (!NFS_CUDA(c, cudaFuncSetAttribute(k_fft<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P::smem))) return false;
  int per_sm = 0;
  if (!NFS_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_fft<L>, P::NT, P::smem))) return false;
  c.fft_grid = std::max(1, per_sm) * std::max(1, c.n_sm);
  return true;
}

template <int L>
static int launch_fft_L(Ctx& c, const FftJob& job, int cls) {
  using P = Plan<L>;
  const long long total = (long long)(job.nf + P::Dr + P::Dc) * P::perStep;
  const int grid = (int)std::min<long long>(c.fft_grid, total);
  ProfScope ps(c, cls);
  if (!NFS_CUDA(c, cudaMemsetAsync(c.fft_cnt, 0, sizeof(unsigned) * (1 + 3 * (size_t)job.nf), c.stream))) return 0;
  if (!NFS_CUDA(c, cudaMemsetAsync(c.sums, 0, sizeof(unsigned long long) * (size_t)job.nf, c.stream))) return 0;
  k_fft<L><<<grid, P::NT, P::smem, c.stream>>>(job);
  NFS_CUDA(c, cudaGetLastError());
  return 1;
}

#define NFS_FFT_SIZES(X) X(32) X(64) X(128) X(256) X(512) X(1024) X(2048) X(4096)

static int launch_fft(Ctx& c, const FftJob& job, int cls) {
  switch (c.W) {
#define X(L) \
  case L: return launch_fft_L<L>(c, job, cls);
    NFS_FFT_SIZES(X)
#undef X
    default: return 0;
  }
}

// once at create: dynamic shared memory of the kernel for this frame size and its persistent grid
bool fft_configure(Ctx& c) {
  switch (c.W) {
#define X(L) \
  case L: return configure_L<L>(c);
    NFS_FFT_SIZES(X)
#undef X
    default: return false;
  }
}

size_t fft_cnt_elems(const Ctx& c) { return 1 + 3 * (size_t)c.B; }

template <int L>
static constexpr int slots_of() { return Plan<L>::slots; }
size_t fft_rowT_elems(const Ctx& c) {
  int slots = kMaxSlots;
  switch (c.W) {
#define X(L) \
  case L: slots = slots_of<L>(); break;
    NFS_FFT_SIZES(X)
#undef X
    default: break;
  }
  return (size_t)slots * (size_t)c.P;
}

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
    if (!NFS_CUDA(c, cudaMemsetAsync(c.sums, 0, sizeof(unsigned long long), c.stream))) return 0;
    int nblk = (int)std::min<int64_t>(592, (npx / 8 + 255) / 256);
    k_frame_sum<<<nblk, 256, 0, c.stream>>>(reinterpret_cast<const uint4*>(frame0), npx / 8, c.sums);
    nblk = (int)std::min<int64_t>(1184, (npx + 1023) / 1024);
    k_make_ref<<<nblk, 256, 0, c.stream>>>(frame0, npx, (float)c.W * (float)c.H, c.sums, c.ref, c.d_flags);
    NFS_CUDA(c, cudaGetLastError());
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
