// nfs_lag.cu — step S5 of the hot path: lag accumulation  A_tau(p) += |F'_{s-tau}(p) - F'_s(p)|^2
// for every new frame s of a batch and every requested lag tau ("only the square
// moduli of FFT differences are evaluated N(N-1)/2 times"; L25 average over the measurement time).
//
// k_lag_tiled (default): a CTA owns 32 consecutive Fourier pixels and one group of lags; it streams
// the batch through shared memory (cp.async, double buffered): a NEW stream (frames s) and an OLD
// stream delayed by the group's lags.  A warp owns up to kG lags: for a run of contiguous lags it
// keeps a rotating register window of the kG most recent OLD frames, so one step costs two LDS.64
// and kG pair-updates; isolated lags take one LDS.64 per update.  fp32 partial sums per batch are
// folded into the fp64 totals once per batch (BASELINE.json north_star (4)).
// k_lag_simple: plain per-pixel kernel through L1/L2, kept as an in-library cross-check.
#include "nfs_common.cuh"

namespace nfs {

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}

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
// tiled kernel
// ------------------------------------------------------------------------------------------------
constexpr int kRowF2 = kTilePx;  // float2 per shared-memory row (one frame, 32 pixels = 256 B)

__host__ __device__ inline int lag_depth(int tau_min, int tau_max) { return (tau_max - tau_min) + 2 * kChunk; }

size_t lag_tiled_smem_bytes(const LagGroup& g) {
  return sizeof(float2) * kRowF2 * (size_t)(lag_depth(g.tau_min, g.tau_max) + kG - 1 + 2 * kChunk);
}

template <int G>
__global__ void __launch_bounds__(kMaxTasks * 32, 2)
    k_lag_tiled(const float2* __restrict__ ring, int R, int64_t P, int64_t t0, int b, const LagTask* __restrict__ tasks,
                const LagGroup* __restrict__ groups, const int32_t* __restrict__ lags, double* __restrict__ totals) {
  extern __shared__ float2 smf[];
  const LagGroup grp = groups[blockIdx.y];
  if ((int64_t)grp.tau_min > t0 + b - 1) return;  // no frame pair of this group exists yet
  const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5;
  const int64_t p0 = (int64_t)blockIdx.x * kTilePx;
  const int DEPTH = lag_depth(grp.tau_min, grp.tau_max);
  float2* OLD = smf;                                   // [DEPTH + G - 1][32]
  float2* NEW = smf + (size_t)(DEPTH + G - 1) * kRowF2;  // [2][kChunk][32]
  const int64_t f_old0 = t0 - grp.tau_max;             // global frame of OLD coordinate e = 0
  const int span1 = grp.tau_max - grp.tau_min;         // OLD rows needed before the first step

  // ---- loaders (all threads): 16 x 16-byte pieces per row ----
  auto load_old = [&](int e_first, int count) {
    for (int idx = tid; idx < count * 16; idx += nthr) {
      const int e = e_first + (idx >> 4), piece = idx & 15;
      const int64_t f = f_old0 + e;
      if (f >= t0 + b) continue;
      const int row = e % DEPTH;
      float2* d0 = OLD + (size_t)row * kRowF2 + piece * 2;
      if (f < 0) {
        const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
        *reinterpret_cast<float4*>(d0) = z;
        if (row < G - 1) *reinterpret_cast<float4*>(d0 + (size_t)DEPTH * kRowF2) = z;
      } else {
        const float2* src = ring + (f % R) * P + p0 + piece * 2;
        cp_async16(d0, src);
        if (row < G - 1) cp_async16(d0 + (size_t)DEPTH * kRowF2, src);
      }
    }
  };
  auto load_new = [&](int chunk) {
    const int j0 = chunk * kChunk;
    float2* dst = NEW + (size_t)(chunk & 1) * kChunk * kRowF2;
    for (int idx = tid; idx < kChunk * 16; idx += nthr) {
      const int r = idx >> 4, piece = idx & 15;
      if (j0 + r >= b) continue;
      cp_async16(dst + (size_t)r * kRowF2 + piece * 2, ring + ((t0 + j0 + r) % R) * P + p0 + piece * 2);
    }
  };

  const int nchunks = (b + kChunk - 1) / kChunk;
  load_old(0, span1 + kChunk);
  load_new(0);
  cp_async_commit();

  // ---- per-warp task state ----
  const bool has_task = warp < grp.ntasks;
  LagTask tk;
  tk.tau0 = tk.cnt = tk.l0 = tk.kind = 0;
  if (has_task) tk = tasks[grp.task0 + warp];
  // acc: fp32 partial sums (re^2 and im^2 lanes).  w: dense task = rotating window of OLD frames;
  // sparse task = w[i].x holds (as int bits) the OLD row of lag i at the current block start.
  float2 acc[G], w[G];
  int o0 = 0;  // dense: OLD row of lag tau0 at the current block start
  int lag_first = 0x3fffffff, lag_last = 0x3fffffff;
#pragma unroll
  for (int g = 0; g < G; ++g) {
    acc[g] = make_float2(0.f, 0.f);
    w[g] = make_float2(0.f, 0.f);
  }
  if (has_task) {
    if (tk.kind == 0) {
      lag_first = tk.tau0;
      lag_last = tk.tau0 + tk.cnt - 1;
      o0 = (grp.tau_max - tk.tau0) % DEPTH;
    } else {
      lag_first = lags[tk.l0];
      lag_last = lags[tk.l0 + tk.cnt - 1];
#pragma unroll
      for (int i = 0; i < G; ++i)
        if (i < tk.cnt) w[i].x = __int_as_float((grp.tau_max - lags[tk.l0 + i]) % DEPTH);
    }
  }

  for (int c = 0; c < nchunks; ++c) {
    if (c + 1 < nchunks) {
      load_old(span1 + (c + 1) * kChunk, kChunk);
      load_new(c + 1);
      cp_async_commit();
      cp_async_wait<1>();
    } else {
      cp_async_wait<0>();
    }
    __syncthreads();

    if (has_task) {
      if (c == 0 && tk.kind == 0) {
        // preload the register window with the G-1 OLD frames preceding the first step
#pragma unroll
        for (int q = 1; q < G; ++q) {
          int e = grp.tau_max - tk.tau0 - q;
          if (e < 0) e = 0;
          w[G - q] = OLD[(size_t)(e % DEPTH) * kRowF2 + lane];
        }
      }
      const float2* newc = NEW + (size_t)(c & 1) * kChunk * kRowF2 + lane;
#pragma unroll 1
      for (int blk = 0; blk < kChunk / G; ++blk) {
        const int jb = c * kChunk + blk * G;
        if (jb >= b) break;
        const int64_t sb = t0 + jb;  // global frame index of the block's first step
        const float2* nb = newc + (size_t)blk * G * kRowF2;
        if (tk.kind == 0) {
          const float2* ob = OLD + (size_t)o0 * kRowF2 + lane;
          if (sb + 2 * G - 1 < (int64_t)lag_first) {
            // neither this block nor the next one holds a valid pair: nothing to keep
          } else if (jb + G <= b && sb >= (int64_t)lag_first + G - 1) {
#pragma unroll
            for (int u = 0; u < G; ++u) {
              const float2 zn = nb[(size_t)u * kRowF2];
              w[u] = ob[(size_t)u * kRowF2];
#pragma unroll
              for (int g = 0; g < G; ++g) upd(acc[g], zn, w[(u - g + G) % G]);
            }
          } else {
#pragma unroll
            for (int u = 0; u < G; ++u) {
              const float2 zn = nb[(size_t)u * kRowF2];
              w[u] = ob[(size_t)u * kRowF2];
              const bool in_batch = jb + u < b;
#pragma unroll
              for (int g = 0; g < G; ++g)
                if (in_batch && sb + u >= (int64_t)lag_first + g) upd(acc[g], zn, w[(u - g + G) % G]);
            }
          }
          o0 += G;
          if (o0 >= DEPTH) o0 -= DEPTH;
        } else {
          if (sb + G - 1 < (int64_t)lag_first) {
            // no valid pair in this block
          } else if (jb + G <= b && sb >= (int64_t)lag_last) {
#pragma unroll
            for (int u = 0; u < G; ++u) {
              const float2 zn = nb[(size_t)u * kRowF2];
#pragma unroll
              for (int i = 0; i < G; ++i)
                if (i < tk.cnt) upd(acc[i], zn, OLD[(size_t)(__float_as_int(w[i].x) + u) * kRowF2 + lane]);
            }
          } else {
#pragma unroll
            for (int u = 0; u < G; ++u) {
              const float2 zn = nb[(size_t)u * kRowF2];
              const bool in_batch = jb + u < b;
#pragma unroll
              for (int i = 0; i < G; ++i)
                if (i < tk.cnt && in_batch && sb + u >= (int64_t)__ldg(&lags[tk.l0 + i]))
                  upd(acc[i], zn, OLD[(size_t)(__float_as_int(w[i].x) + u) * kRowF2 + lane]);
            }
          }
#pragma unroll
          for (int i = 0; i < G; ++i) {
            int o = __float_as_int(w[i].x) + G;
            if (o >= DEPTH) o -= DEPTH;
            w[i].x = __int_as_float(o);
          }
        }
      }
    }
    __syncthreads();
  }

  if (has_task) {
    const int64_t p = p0 + lane;
#pragma unroll
    for (int g = 0; g < G; ++g)
      if (g < tk.cnt) {
        double* dst = totals + (int64_t)(tk.l0 + g) * P + p;
        *dst += (double)(acc[g].x + acc[g].y);
      }
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
  k_lag_tiled<kG><<<grid, kMaxTasks * 32, smem, c.stream>>>(c.ring, c.R, c.P, t0, b, c.d_tasks, c.d_groups, c.d_lags,
                                                          c.totals);
  return 1;
}

}  // namespace nfs
