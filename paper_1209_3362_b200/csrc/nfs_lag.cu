// nfs_lag.cu — step S5 of the hot path: lag accumulation  A_tau(p) += |F'_{s-tau}(p) - F'_s(p)|^2
// for every new frame s of a batch and every requested lag tau ("only the square
// moduli of FFT differences are evaluated N(N-1)/2 times"; L25 average over the measurement time).
//
// k_lag_tiled (default): a CTA owns 32 consecutive Fourier pixels and one group of lags; a producer
// warp streams the batch through shared memory with bulk copies (cp.async.bulk + mbarrier, 3 stages):
// a NEW stream (frames s) and an OLD stream delayed by the group's lags.  A consumer warp owns up to
// kG lags: for a run of contiguous lags it keeps a rotating register window of the kG most recent OLD
// frames, so one step costs two LDS.64 and kG pair-updates (packed sub.f32x2 + fma.rn.f32x2: two issue
// slots per update); isolated lags take one LDS.64 per update.  fp32 partial sums per batch are
// folded into the fp64 totals once per batch (BASELINE.json north_star (4)).
// k_lag_simple: plain per-pixel kernel through L1/L2, kept as an in-library cross-check.
#include "nfs_common.cuh"

namespace nfs {

__device__ __forceinline__ void upd(float2& acc, float2 zn, float2 zo) {
  const float dx = zn.x - zo.x, dy = zn.y - zo.y;
  acc.x = fmaf(dx, dx, acc.x);
  acc.y = fmaf(dy, dy, acc.y);
}

// ------------------------------------------------------------------------------------------------
// I accumulators: I2 += sum |F'_s|^2, I1 += sum F'_s over the batch (R9; static spectrum
// is rebuilt at finalize as <|F'+F_r|^2>).  One thread per pixel, fp32 partials folded every 64 steps.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_accum_I(const float2* __restrict__ ring, int R, int64_t P, int64_t t0, int b,
                                                 double* __restrict__ I2, double2* __restrict__ I1) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  double d2 = 0.0, dx = 0.0, dy = 0.0;
  int slot = (int)(t0 % R);
  for (int j0 = 0; j0 < b; j0 += 64) {
    float a2 = 0.f, ax = 0.f, ay = 0.f;
    const int je = min(b, j0 + 64);
    for (int j = j0; j < je; ++j) {
      const float2 z = __ldcs(&ring[(int64_t)slot * P + p]);
      a2 = fmaf(z.x, z.x, fmaf(z.y, z.y, a2));
      ax += z.x;
      ay += z.y;
      if (++slot == R) slot = 0;
    }
    d2 += (double)a2;
    dx += (double)ax;
    dy += (double)ay;
  }
  I2[p] += d2;
  double2 v = I1[p];
  v.x += dx;
  v.y += dy;
  I1[p] = v;
}

// ------------------------------------------------------------------------------------------------
// plain kernel: thread = (pixel, 8 consecutive lag indices); grid (ceil(P/128), ceil(n_lags/8))
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_lag_simple(const float2* __restrict__ ring, int R, int64_t P, int64_t t0, int b,
                                                    const int32_t* __restrict__ lags, int n_lags,
                                                    double* __restrict__ totals) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  const int l0 = blockIdx.y * 8;
  int tau[8];
  float2 acc[8];
#pragma unroll
  for (int g = 0; g < 8; ++g) {
    tau[g] = (l0 + g < n_lags) ? lags[l0 + g] : 0x7fffffff;
    acc[g] = make_float2(0.f, 0.f);
  }
  for (int j = 0; j < b; ++j) {
    const int64_t s = t0 + j;
    const float2 zn = ring[(s % R) * P + p];
#pragma unroll
    for (int g = 0; g < 8; ++g) {
      if (s >= tau[g]) {
        const float2 zo = ring[((s - tau[g]) % R) * P + p];
        upd(acc[g], zn, zo);
      }
    }
  }
#pragma unroll
  for (int g = 0; g < 8; ++g)
    if (l0 + g < n_lags) totals[(int64_t)(l0 + g) * P + p] += (double)(acc[g].x + acc[g].y);
}

// ------------------------------------------------------------------------------------------------
// tiled kernel: warp-specialised.  Warp 0 = producer (bulk copies global -> shared, completion on
// mbarriers), warps 1..ntasks = consumers (one lag task each).  Shared memory:
//   OLD ring  [DEPTH + G - 1][32] float2   frames s - tau for the group's lags; row e holds global
//             frame f_old0 + e at row e % DEPTH (rows 0..G-2 duplicated behind the end so that a
//             block of G consecutive rows never wraps)
//   NEW       [kStages][kChunk][32] float2 the batch's own frames
// Chunk c (kChunk time steps) lives in stage c % kStages; full[stage] counts the producer lanes'
// arrivals + the bytes of their copies, empty[stage] counts the consumer warps that are done with it.
// ------------------------------------------------------------------------------------------------
constexpr int kRowF2 = kTilePx;                 // float2 per shared-memory row (one frame, 32 pixels = 256 B)
constexpr unsigned kRowBytes = kRowF2 * 8u;
constexpr int kStages = 3;

__host__ __device__ inline int lag_depth(int tau_min, int tau_max) { return (tau_max - tau_min) + kStages * kChunk; }

size_t lag_tiled_smem_bytes(const LagGroup& g) {
  return 64 + sizeof(float2) * kRowF2 * (size_t)(lag_depth(g.tau_min, g.tau_max) + kG - 1 + kStages * kChunk);
}

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
// 1-D bulk copy global -> shared (TMA engine, SASS UBLKCP); completes `bytes` on the mbarrier
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// packed fp32x2 arithmetic (SASS FADD2 / FFMA2): one issue slot for both components of a complex number
typedef unsigned long long f2x;
__device__ __forceinline__ f2x sub2(f2x a, f2x b) {
  f2x r;
  asm("sub.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ f2x fma2(f2x a, f2x b, f2x c) {
  f2x r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
__device__ __forceinline__ void upd2(f2x& acc, f2x zn, f2x zo) {
  const f2x d = sub2(zn, zo);
  acc = fma2(d, d, acc);
}
__device__ __forceinline__ float f2x_sum(f2x v) {
  return __uint_as_float((unsigned)(v & 0xffffffffull)) + __uint_as_float((unsigned)(v >> 32));
}

template <int G>
__global__ void __launch_bounds__((kMaxTasks + 1) * 32, 2)
    k_lag_tiled(const float2* __restrict__ ring, int R, int64_t P, int64_t t0, int b, const LagTask* __restrict__ tasks,
                const LagGroup* __restrict__ groups, const int32_t* __restrict__ lags, double* __restrict__ totals) {
  extern __shared__ __align__(128) unsigned char smraw[];
  const LagGroup grp = groups[blockIdx.y];
  if ((int64_t)grp.tau_min > t0 + b - 1) return;  // no frame pair of this group exists yet
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t p0 = (int64_t)blockIdx.x * kTilePx;
  const int DEPTH = lag_depth(grp.tau_min, grp.tau_max);
  uint64_t* full = reinterpret_cast<uint64_t*>(smraw);      // [kStages]
  uint64_t* empty = full + kStages;                         // [kStages]
  f2x* OLD = reinterpret_cast<f2x*>(smraw + 64);            // [DEPTH + G - 1][32]
  f2x* NEW = OLD + (size_t)(DEPTH + G - 1) * kRowF2;        // [kStages][kChunk][32]
  const int span1 = grp.tau_max - grp.tau_min;              // OLD rows needed before the first step
  const int nchunks = (b + kChunk - 1) / kChunk;

  if (tid == 0) {
    for (int s = 0; s < kStages; ++s) {
      mbar_init(&full[s], 32);
      mbar_init(&empty[s], (unsigned)grp.ntasks);
    }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();

  if (warp == 0) {
    // ------------------------------- producer -------------------------------
    const int64_t f_old0 = t0 - grp.tau_max;  // global frame of OLD coordinate e = 0
    const float2* tile = ring + p0;
    for (int c = 0; c < nchunks; ++c) {
      const int st = c % kStages;
      if (c >= kStages) mbar_wait(&empty[st], ((c / kStages) - 1) & 1);
      // OLD rows of this chunk: the first chunk also brings the span1 rows preceding the first step
      const int e_first = c == 0 ? 0 : span1 + c * kChunk;
      const int count = c == 0 ? span1 + kChunk : kChunk;
      unsigned bytes = 0;
      for (int i = lane; i < count; i += 32) {
        const int e = e_first + i;
        const int64_t f = f_old0 + e;
        if (f < 0 || f >= t0 + b) continue;  // before the first frame / beyond this batch: never used
        const int row = e % DEPTH;
        const float2* src = tile + (f % R) * P;
        bulk_g2s(OLD + (size_t)row * kRowF2, src, kRowBytes, &full[st]);
        bytes += kRowBytes;
        if (row < G - 1) {
          bulk_g2s(OLD + (size_t)(row + DEPTH) * kRowF2, src, kRowBytes, &full[st]);
          bytes += kRowBytes;
        }
      }
      if (lane < kChunk) {
        const int j = c * kChunk + lane;
        if (j < b) {
          bulk_g2s(NEW + ((size_t)st * kChunk + lane) * kRowF2, tile + ((t0 + j) % R) * P, kRowBytes, &full[st]);
          bytes += kRowBytes;
        }
      }
      mbar_arrive_expect_tx(&full[st], bytes);
    }
    return;
  }

  // ------------------------------- consumers -------------------------------
  if (warp > grp.ntasks) return;
  const LagTask tk = tasks[grp.task0 + warp - 1];
  // acc: fp32 partial sums (re^2 and im^2 lanes, packed).  w: dense task = rotating window of OLD
  // frames; sparse task = low word of w[i] holds the OLD row of lag i at the current block start.
  f2x acc[G], w[G];
#pragma unroll
  for (int g = 0; g < G; ++g) acc[g] = 0ull, w[g] = 0ull;
  // validity in batch-relative steps: pair (j, lag) exists iff j >= lag - t0
  const int64_t dt = (int64_t)tk.tau0 - t0;
  int jfirst, jlast, o0 = 0;
  if (tk.kind == 0) {
    jfirst = (int)max(dt, (int64_t)-(1 << 24));
    jlast = jfirst + tk.cnt - 1;
    o0 = (grp.tau_max - tk.tau0) % DEPTH;
  } else {
    jfirst = (int)max((int64_t)lags[tk.l0] - t0, (int64_t)-(1 << 24));
    jlast = (int)max((int64_t)lags[tk.l0 + tk.cnt - 1] - t0, (int64_t)-(1 << 24));
#pragma unroll
    for (int i = 0; i < G; ++i)
      if (i < tk.cnt) w[i] = (f2x)(unsigned)((grp.tau_max - lags[tk.l0 + i]) % DEPTH);
  }

  for (int c = 0; c < nchunks; ++c) {
    const int st = c % kStages;
    mbar_wait(&full[st], (c / kStages) & 1);

    if (c == 0 && tk.kind == 0) {
      // preload the register window with the G-1 OLD frames preceding the first step
#pragma unroll
      for (int q = 1; q < G; ++q) {
        int e = grp.tau_max - tk.tau0 - q;
        if (e < 0) e = 0;
        w[G - q] = OLD[(size_t)(e % DEPTH) * kRowF2 + lane];
      }
    }
    const f2x* newc = NEW + (size_t)st * kChunk * kRowF2 + lane;
#pragma unroll 1
    for (int blk = 0; blk < kChunk / G; ++blk) {
      const int jb = c * kChunk + blk * G;  // batch-relative index of the block's first step
      if (jb >= b) break;
      const f2x* nb = newc + (size_t)blk * G * kRowF2;
      if (tk.kind == 0) {
        const f2x* ob = OLD + (size_t)o0 * kRowF2 + lane;
        if (jb + 2 * G - 1 < jfirst) {
          // neither this block nor the next one holds a valid pair: nothing to keep
        } else if (jb + G <= b && jb >= jlast) {
#pragma unroll
          for (int u = 0; u < G; ++u) {
            const f2x zn = nb[(size_t)u * kRowF2];
            w[u] = ob[(size_t)u * kRowF2];
#pragma unroll
            for (int g = 0; g < G; ++g) upd2(acc[g], zn, w[(u - g + G) % G]);
          }
        } else {
#pragma unroll
          for (int u = 0; u < G; ++u) {
            const f2x zn = nb[(size_t)u * kRowF2];
            w[u] = ob[(size_t)u * kRowF2];
            const bool in_batch = jb + u < b;
#pragma unroll
            for (int g = 0; g < G; ++g)
              if (in_batch && g < tk.cnt && jb + u >= jfirst + g) upd2(acc[g], zn, w[(u - g + G) % G]);
          }
        }
        o0 += G;
        if (o0 >= DEPTH) o0 -= DEPTH;
      } else {
        if (jb + G - 1 < jfirst) {
          // no valid pair in this block
        } else if (jb + G <= b && jb >= jlast) {
#pragma unroll
          for (int u = 0; u < G; ++u) {
            const f2x zn = nb[(size_t)u * kRowF2];
#pragma unroll
            for (int i = 0; i < G; ++i)
              if (i < tk.cnt) upd2(acc[i], zn, OLD[(size_t)((unsigned)w[i] + u) * kRowF2 + lane]);
          }
        } else {
#pragma unroll
          for (int u = 0; u < G; ++u) {
            const f2x zn = nb[(size_t)u * kRowF2];
            const bool in_batch = jb + u < b;
#pragma unroll
            for (int i = 0; i < G; ++i)
              if (i < tk.cnt && in_batch && (int64_t)(jb + u) >= (int64_t)__ldg(&lags[tk.l0 + i]) - t0)
                upd2(acc[i], zn, OLD[(size_t)((unsigned)w[i] + u) * kRowF2 + lane]);
          }
        }
#pragma unroll
        for (int i = 0; i < G; ++i) {
          unsigned o = (unsigned)w[i] + G;
          if (o >= (unsigned)DEPTH) o -= DEPTH;
          w[i] = (f2x)o;
        }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[st]);
  }

  const int64_t p = p0 + lane;
#pragma unroll
  for (int g = 0; g < G; ++g)
    if (g < tk.cnt) {
      double* dst = totals + (int64_t)(tk.l0 + g) * P + p;
      *dst += (double)f2x_sum(acc[g]);
    }
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
int launch_accum_I(Ctx& c, int64_t t0, int b) {
  ProfScope ps(c, kKAccI);
  k_accum_I<<<(unsigned)((c.P + 255) / 256), 256, 0, c.stream>>>(c.ring, c.R, c.P, t0, b, c.I2, c.I1);
  return 1;
}

int launch_lag_simple(Ctx& c, int64_t t0, int b) {
  dim3 grid((unsigned)((c.P + 127) / 128), (unsigned)((c.n_lags + 7) / 8));
  ProfScope ps(c, kKLag);
  k_lag_simple<<<grid, 128, 0, c.stream>>>(c.ring, c.R, c.P, t0, b, c.d_lags, c.n_lags, c.totals);
  return 1;
}

int launch_lag_tiled(Ctx& c, int64_t t0, int b) {
  size_t smem = 0;
  for (const LagGroup& g : c.groups) {
    size_t s = lag_tiled_smem_bytes(g);
    if (s > smem) smem = s;
  }
  static_assert(kChunk % kG == 0, "chunk must hold whole blocks of kG steps");
  cudaFuncSetAttribute(k_lag_tiled<kG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  dim3 grid((unsigned)(c.P / kTilePx), (unsigned)c.groups.size());
  ProfScope ps(c, kKLag);
  k_lag_tiled<kG><<<grid, (kMaxTasks + 1) * 32, smem, c.stream>>>(c.ring, c.R, c.P, t0, b, c.d_tasks, c.d_groups, c.d_lags,
                                                          c.totals);
  return 1;
}

}  // namespace nfs
