// nfs_lag.cu — step S5 of the hot path: lag accumulation  A_tau(p) += |F'_{s-tau}(p) - F'_s(p)|^2
// for every new frame s of a batch and every requested lag tau ("only the square
// moduli of FFT differences are evaluated N(N-1)/2 times"; L25 average over the measurement time).
//
// k_lag_tiled (default): a CTA works on 32 consecutive Fourier pixels and one group of lags at a time; a
// producer warp streams the batch through shared memory with TMA tensor copies (cp.async.bulk.tensor +
// mbarrier): a NEW stream (frames s) and an OLD stream delayed by the group's lags.  A consumer warp owns up to
// kG lags: for a run of contiguous lags it keeps a rotating register window of the kG most recent OLD
// frames, so one step costs two LDS.64 and kG pair-updates (packed sub.f32x2 + fma.rn.f32x2: two issue
// slots per update); isolated lags take one LDS.64 per update.  fp32 partial sums are folded into the fp64
// totals every kFoldChunks chunks and at the end of a tile (BASELINE.json north_star (4)).  One warp of the
// lightest group also adds the batch to the I sums (sum |F'|^2, sum F').
// Two launch shapes (template parameter PERS, chosen per batch by launch_lag_tiled): one CTA per (pixel tile,
// lag group), or persistent CTAs that claim the pixel tiles of their group and keep the pipeline full across
// tiles.  Results do not depend on the shape.
// k_lag_simple: plain per-pixel kernel through L1/L2, kept as an in-library cross-check.
#include <algorithm>

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
// tiled kernel: warp-specialised.  Warps 0..kMaxTasks-1 = consumers (one lag task each, placed by the
// plan so that the four SM sub-partitions carry equal work), the last warp = producer (highest warp
// id: first in the issue arbiter, so loads are never starved by the math warps).
// Time is cut into chunks of kChunk = 2*kG steps.  Shared memory, in rows of 32 pixels (256 B):
//   OLD  [(NSLOT + 1) * kChunk]  ring of NSLOT = LEAD + stages chunk slots; OLD row e holds frame
//                                E0 + e, E0 = t0 - tau_min - LEAD*kChunk, at row e % (NSLOT*kChunk); the
//                                last kChunk rows duplicate slot 0 so kG consecutive rows never wrap
//   NEW  [stages * kChunk]       the batch's own frames, chunk c in stage c % stages
// full[stage]: the producer's arrival + the bytes of its copies for one pipeline step; empty[stage]: the
// consumer warps.  One tile per CTA: step = consumer chunk c (NEW chunk c, OLD chunk c + LEAD; chunk 0 also
// brings OLD chunks 0..LEAD-1).  Persistent: every tile has LEAD prologue steps that bring one OLD chunk each,
// then one step per chunk (OLD chunk j, NEW chunk j - LEAD); steps and ring slots are numbered through all the
// tiles of the CTA, so the next tile's window streams in while the last chunks of the current one are consumed.
// `stages` (2..kMaxStages) is chosen at create from the shared memory the widest lag group leaves, so
// that the producer runs several chunks (each ~3 us of math) ahead of the HBM/L2 latency.
// A chunk of frames that is contiguous in the HBM ring is one 2-D TMA box (cp.async.bulk.tensor,
// 32 pixels x kChunk ring slots); a chunk that straddles the ring's wrap-around or starts before the
// first frame falls back to one 256-byte bulk copy per row.
// ------------------------------------------------------------------------------------------------
constexpr int kRowF2 = kTilePx;                 // float2 per shared-memory row (one frame, 32 pixels = 256 B)
constexpr unsigned kRowBytes = kRowF2 * 8u;

__host__ __device__ inline int lag_lead(int tau_min, int tau_max) { return (tau_max - tau_min + kChunk - 1) / kChunk; }

static size_t lag_smem_bytes(int tau_min, int tau_max, int stages) {
  const int nslot = lag_lead(tau_min, tau_max) + stages;
  return 128 + sizeof(float2) * kRowF2 * (size_t)((nslot + 1) * kChunk + stages * kChunk);
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
#ifndef NFS_LAG_PROD_HINT_NS
#define NFS_LAG_PROD_HINT_NS 20000
#endif
// producer side: same wait with a suspend-time hint, so that the idle warp does not burn issue slots
__device__ __forceinline__ void mbar_wait_relaxed(uint64_t* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAITR_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n"
      "@p bra DONER_%=;\n"
      "bra WAITR_%=;\n"
      "DONER_%=:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity), "r"((unsigned)NFS_LAG_PROD_HINT_NS)
      : "memory");
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
// 2-D tensor copy global -> shared (SASS UTMALDG): box = 32 pixels (64 floats) x kChunk ring slots
__device__ __forceinline__ void tma_box_g2s(void* dst, const CUtensorMap* tmap, int c0, int c1, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n" ::"r"(
          smem_u32(dst)),
      "l"(tmap), "r"(c0), "r"(c1), "r"(smem_u32(bar))
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
__device__ __forceinline__ f2x add2(f2x a, f2x b) {
  f2x r;
  asm("add.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ void upd2(f2x& acc, f2x zn, f2x zo) {
  const f2x d = sub2(zn, zo);
  acc = fma2(d, d, acc);
}
__device__ __forceinline__ float f2x_sum(f2x v) {
  return __uint_as_float((unsigned)(v & 0xffffffffull)) + __uint_as_float((unsigned)(v >> 32));
}

// producer: bring frames f0 .. f0+kChunk-1 of this pixel tile into shared rows dst (and dup, if given).
// Returns the bytes this lane's copies will complete on the barrier.
__device__ __forceinline__ unsigned load_chunk(const CUtensorMap* tmap, const float2* __restrict__ ring, int R, int64_t P,
                                               int64_t p0, int64_t f0, f2x* dst, f2x* dup, uint64_t* bar, int lane) {
  const int s0 = (int)(((f0 % R) + R) % R);
  if (f0 >= 0 && s0 + kChunk <= R) {
    if (lane != 0) return 0u;
    tma_box_g2s(dst, tmap, (int)(2 * p0), s0, bar);
    if (dup) tma_box_g2s(dup, tmap, (int)(2 * p0), s0, bar);
    return (dup ? 2u : 1u) * kChunk * kRowBytes;
  }
  unsigned bytes = 0;
  if (lane < kChunk) {
    const int64_t f = f0 + lane;
    if (f >= 0) {  // rows before the first frame are never used
      const float2* src = ring + (f % R) * P + p0;
      bulk_g2s(dst + (size_t)lane * kRowF2, src, kRowBytes, bar);
      bytes = kRowBytes;
      if (dup) {
        bulk_g2s(dup + (size_t)lane * kRowF2, src, kRowBytes, bar);
        bytes += kRowBytes;
      }
    }
  }
  return bytes;
}

// One block of kG steps of a dense task with exactly CNT lags: step u loads the new frame and the one
// OLD frame entering the rotating window (2 LDS.64), then CNT pair updates out of registers.
template <int CNT>
__device__ __forceinline__ void dense_block(f2x (&acc)[kG], f2x (&w)[kG], const f2x* nb, const f2x* ob) {
#pragma unroll
  for (int u = 0; u < kG; ++u) {
    const f2x zn = nb[(size_t)u * kRowF2];
    w[u] = ob[(size_t)u * kRowF2];
#pragma unroll
    for (int g = 0; g < CNT; ++g) upd2(acc[g], zn, w[(u - g + kG) % kG]);
  }
}
// ---- whole chunks (kChunk = kChunk/kG blocks) in which every pair of every step exists: the common case ----
template <int CNT>
__device__ __forceinline__ void dense_chunk(f2x (&acc)[kG], f2x (&w)[kG], const f2x* newc, const f2x* oldl, int& o0,
                                            int DEPTH) {
#pragma unroll 1
  for (int blk = 0; blk < kChunk / kG; ++blk) {
    dense_block<CNT>(acc, w, newc + (size_t)blk * kG * kRowF2, oldl + (size_t)o0 * kRowF2);
    o0 += kG;
    if (o0 >= DEPTH) o0 -= DEPTH;
  }
}
__device__ __forceinline__ void dense_chunk_dispatch(int cnt, f2x (&acc)[kG], f2x (&w)[kG], const f2x* newc, const f2x* oldl,
                                                     int& o0, int DEPTH) {
  switch (cnt) {  // warp-uniform; the plan makes dense tasks of kDenseMin..kG lags
    case 12: dense_chunk<12>(acc, w, newc, oldl, o0, DEPTH); break;
    case 11: dense_chunk<11>(acc, w, newc, oldl, o0, DEPTH); break;
    case 10: dense_chunk<10>(acc, w, newc, oldl, o0, DEPTH); break;
    case 9: dense_chunk<9>(acc, w, newc, oldl, o0, DEPTH); break;
    case 8: dense_chunk<8>(acc, w, newc, oldl, o0, DEPTH); break;
    case 7: dense_chunk<7>(acc, w, newc, oldl, o0, DEPTH); break;
    default: dense_chunk<kG>(acc, w, newc, oldl, o0, DEPTH); break;  // 13 (shorter runs: surplus lags are discarded)
  }
}
template <int CNT>
__device__ __forceinline__ void sparse_chunk(f2x (&acc)[kG], f2x (&w)[kG], const f2x* newc, const f2x* oldl, int DEPTH) {
#pragma unroll 1
  for (int blk = 0; blk < kChunk / kG; ++blk) {
    const f2x* nb = newc + (size_t)blk * kG * kRowF2;
#pragma unroll
    for (int u = 0; u < kG; ++u) {
      const f2x zn = nb[(size_t)u * kRowF2];
#pragma unroll
      for (int i = 0; i < CNT; ++i) upd2(acc[i], zn, oldl[(size_t)((unsigned)w[i] + u) * kRowF2]);
    }
#pragma unroll
    for (int i = 0; i < CNT; ++i) {
      unsigned o = (unsigned)w[i] + kG;
      if (o >= (unsigned)DEPTH) o -= DEPTH;
      w[i] = (f2x)o;
    }
  }
}
__device__ __forceinline__ void sparse_chunk_dispatch(int cnt, f2x (&acc)[kG], f2x (&w)[kG], const f2x* newc, const f2x* oldl,
                                                      int DEPTH) {
  switch (cnt) {
    case 0: break;  // a task that only accumulates the I sums
    case 1: sparse_chunk<1>(acc, w, newc, oldl, DEPTH); break;
    case 2: sparse_chunk<2>(acc, w, newc, oldl, DEPTH); break;
    case 3: sparse_chunk<3>(acc, w, newc, oldl, DEPTH); break;
    case 4: sparse_chunk<4>(acc, w, newc, oldl, DEPTH); break;
    case 5: sparse_chunk<5>(acc, w, newc, oldl, DEPTH); break;
    default: sparse_chunk<kSparseMax>(acc, w, newc, oldl, DEPTH); break;  // the plan makes lag lists of <= kSparseMax
  }
}

// One block of a lag-list task with exactly CNT lags in which some pairs do not exist (warm-up: the OLD
// frame would precede the first frame; or the batch's ragged tail): pair (step u, lag i) is counted iff
// u >= u0_i = lag_i - (frame number of step 0), and u < ns.
template <int CNT>
__device__ __forceinline__ void sparse_masked(int ns, f2x (&acc)[kG], const f2x (&w)[kG], const f2x* nb, const f2x* oldl,
                                              const int* my_lags, int64_t frame0) {
  int u0[CNT];
#pragma unroll
  for (int i = 0; i < CNT; ++i) u0[i] = (int)min((int64_t)99, max((int64_t)0, (int64_t)my_lags[i] - frame0));
#pragma unroll
  for (int u = 0; u < kG; ++u) {
    if (u < ns) {
      const f2x zn = nb[(size_t)u * kRowF2];
#pragma unroll
      for (int i = 0; i < CNT; ++i)
        if (u >= u0[i]) upd2(acc[i], zn, oldl[(size_t)((unsigned)w[i] + u) * kRowF2]);
    }
  }
}
__device__ __forceinline__ void sparse_masked_dispatch(int cnt, int ns, f2x (&acc)[kG], const f2x (&w)[kG], const f2x* nb,
                                                       const f2x* oldl, const int* my_lags, int64_t frame0) {
  switch (cnt) {
    case 0: break;
    case 1: sparse_masked<1>(ns, acc, w, nb, oldl, my_lags, frame0); break;
    case 2: sparse_masked<2>(ns, acc, w, nb, oldl, my_lags, frame0); break;
    case 3: sparse_masked<3>(ns, acc, w, nb, oldl, my_lags, frame0); break;
    case 4: sparse_masked<4>(ns, acc, w, nb, oldl, my_lags, frame0); break;
    case 5: sparse_masked<5>(ns, acc, w, nb, oldl, my_lags, frame0); break;
    default: sparse_masked<kSparseMax>(ns, acc, w, nb, oldl, my_lags, frame0); break;
  }
}

template <bool PERS, bool SKIP>
__global__ void __launch_bounds__((kMaxTasks + 1) * 32, kLagMinBlocks)
    k_lag_tiled(const __grid_constant__ CUtensorMap tmap, const float2* __restrict__ ring, int R, int64_t P,
                int64_t t0_batch, int b_batch, int ngroups, int stages, const LagTask* __restrict__ tasks, const LagGroup* __restrict__ groups,
                const int32_t* __restrict__ lags, double* __restrict__ totals, double* __restrict__ I2,
                double2* __restrict__ I1, int ntiles, int* __restrict__ claim) {
  constexpr int G = kG;
  static_assert(kChunk % G == 0 && kChunk <= 32, "a chunk is a whole number of G-step blocks, one lane per row");
  static_assert(kSparseMax == 6, "sparse_chunk_dispatch lists cases 0..5 and the default");
  static_assert(kMaxTasks <= 16 && kMaxTasks % 4 == 0, "warp_task[16], whole sub-partition rounds");
  extern __shared__ __align__(128) unsigned char smraw[];
  __shared__ int s_lags[kMaxTasks * kG];  // the lags of each sparse task, for the warm-up path
  __shared__ int s_tile[kMaxStages];      // tile of the item whose first step uses this stage, or -1: no more work
  // persistent launch: group gi owns CTAs [cta0, cta0 + nctas), which claim the group's pixel tiles one after
  // the other (claim[gi], zeroed before the launch) and run through them without draining the shared-memory
  // pipeline.  One-tile launch: CTA = (tile, group), the groups of a tile side by side (they share L2 lines).
  int gi = 0;
  if constexpr (PERS) {
    while (gi + 1 < ngroups && (int)blockIdx.x >= groups[gi].cta0 + groups[gi].nctas) ++gi;
  } else {
    gi = blockIdx.x % ngroups;
  }
  const LagGroup& grp = groups[gi];
  const int tau_min = grp.tau_min, tau_max = grp.tau_max;
  // no frame pair of this group exists yet (the group that accumulates the I sums always runs)
  if (grp.flags == 0 && (int64_t)tau_min > t0_batch + b_batch - 1) return;
  // SKIP (launched only while some group's smallest lag still reaches back before frame 0): such a group skips
  // the whole chunks in which it has no pair, i.e. it works on the batch cut at the front (the I sums need every
  // frame: that group keeps the whole batch).  Otherwise t0 and b stay kernel parameters (no registers).
  int64_t t0 = t0_batch;
  int b = b_batch;
  if constexpr (SKIP) {
    if (grp.flags == 0 && (int64_t)tau_min > t0) {
      const int skip = (int)(((int64_t)tau_min - t0) / kChunk) * kChunk;
      t0 += skip;
      b -= skip;
    }
  }
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int LEAD = lag_lead(tau_min, tau_max);
  const int NSLOT = LEAD + stages;
  const int DEPTH = NSLOT * kChunk;
  uint64_t* full = reinterpret_cast<uint64_t*>(smraw);      // [kMaxStages]
  uint64_t* empty = full + kMaxStages;                      // [kMaxStages]
  static_assert(2 * kMaxStages * 8 <= 128, "barriers fit the 128-byte header");
  f2x* OLD = reinterpret_cast<f2x*>(smraw + 128);           // [(NSLOT + 1) * kChunk][32]
  f2x* NEW = OLD + (size_t)(NSLOT + 1) * kChunk * kRowF2;   // [stages][kChunk][32]
  const int nchunks = (b + kChunk - 1) / kChunk;
  // One item (pixel tile) = LEAD prologue steps that only bring OLD chunks (the window), then nchunks steps that
  // bring OLD chunk j and NEW chunk j - LEAD and are consumed.  Steps are numbered through all items of the
  // CTA: step v uses pipeline stage v % stages and puts its OLD chunk into ring slot v % NSLOT, which held the
  // OLD chunk of step v - NSLOT = v - LEAD - stages, last read by the consumers at step v - stages.
  const int V = nchunks + LEAD;

  if (tid == 0) {
    const unsigned nt = (unsigned)grp.ntasks;
    for (int s = 0; s < stages; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], nt);
    }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();

  if (warp == kMaxTasks) {
    // ------------------------------- producer -------------------------------
    const int64_t E0 = t0 - tau_min - (int64_t)LEAD * kChunk;  // frame held by row 0 of an item's OLD chunk 0
    int st = 0, slot = 0;
    unsigned ph = 0;  // parity of this stage's current use
    if constexpr (PERS) {
      for (;;) {
        int tile = 0;
        if (lane == 0) tile = atomicAdd(&claim[gi], 1);
        tile = __shfl_sync(0xffffffffu, tile, 0);
        if (tile >= ntiles) {  // tell the consumers; nothing is loaded for this step
          mbar_wait_relaxed(&empty[st], ph ^ 1u);
          if (lane == 0) {
            s_tile[st] = -1;
            mbar_arrive(&full[st]);
          }
          break;
        }
        const int64_t p0 = (int64_t)tile * kTilePx;
        for (int j = 0; j < V; ++j) {
          mbar_wait_relaxed(&empty[st], ph ^ 1u);  // passes at once on the first use of a stage
          if (j == 0 && lane == 0) s_tile[st] = tile;  // ordered before the consumers' read by the arrive below
          f2x* dst = OLD + (size_t)slot * kChunk * kRowF2;
          f2x* dup = slot == 0 ? OLD + (size_t)NSLOT * kChunk * kRowF2 : nullptr;
          unsigned bytes = load_chunk(&tmap, ring, R, P, p0, E0 + (int64_t)j * kChunk, dst, dup, &full[st], lane);
          if (j >= LEAD)
            bytes += load_chunk(&tmap, ring, R, P, p0, t0 + (int64_t)(j - LEAD) * kChunk,
                                NEW + (size_t)st * kChunk * kRowF2, nullptr, &full[st], lane);
          bytes = __reduce_add_sync(0xffffffffu, bytes);
          if (lane == 0) mbar_arrive_expect_tx(&full[st], bytes);
          if (++st == stages) st = 0, ph ^= 1u;
          if (++slot == NSLOT) slot = 0;
        }
      }
    } else {
      // one pixel tile: the whole window (OLD chunks 0..LEAD) comes with the first chunk, no prologue steps
      const int64_t p0 = (int64_t)(blockIdx.x / ngroups) * kTilePx;
      for (int c = 0; c < nchunks; ++c) {
        if (c >= stages) mbar_wait_relaxed(&empty[st], ph ^ 1u);
        unsigned bytes = load_chunk(&tmap, ring, R, P, p0, t0 + (int64_t)c * kChunk, NEW + (size_t)st * kChunk * kRowF2,
                                    nullptr, &full[st], lane);
        for (int m = (c == 0 ? 0 : c + LEAD); m <= c + LEAD; ++m) {
          f2x* dst = OLD + (size_t)slot * kChunk * kRowF2;
          f2x* dup = slot == 0 ? OLD + (size_t)NSLOT * kChunk * kRowF2 : nullptr;
          bytes += load_chunk(&tmap, ring, R, P, p0, E0 + (int64_t)m * kChunk, dst, dup, &full[st], lane);
          if (++slot == NSLOT) slot = 0;
        }
        bytes = __reduce_add_sync(0xffffffffu, bytes);
        if (lane == 0) mbar_arrive_expect_tx(&full[st], bytes);
        if (++st == stages) st = 0, ph ^= 1u;
      }
    }
    return;
  }

  // ------------------------------- consumers -------------------------------
  const int tix = grp.warp_task[warp];
  if (tix < 0) return;
  const LagTask tk = tasks[grp.task0 + tix];
  const bool dense = (tk.kind & 1) == 0;
  const bool doI = (tk.kind & 2) != 0;  // this warp also accumulates I2 += |F'_s|^2, I1 += F'_s (group 0 only)
  const int cnt = tk.cnt;
  f2x i2 = 0ull, i1 = 0ull;             // fp32 partials of the batch (<= 1024 terms, like acc)
  // acc: fp32 partial sums (re^2 and im^2 lanes, packed).  Dense task: w = rotating window of the G most
  // recent OLD frames.  Sparse task: the low word of w[i] holds the OLD row of lag i at the block start.
  f2x acc[G], w[G];
#pragma unroll
  for (int g = 0; g < G; ++g) acc[g] = 0ull, w[g] = 0ull;
  // OLD row (before the ring modulo) of the frame that lag tau pairs with step j:  j + offbase - tau
  const int offbase = LEAD * kChunk + tau_min;
  int o0 = 0;           // dense: ring row of frame (t0 + jb - tau0) at the current block start
  bool wvalid = false;  // dense: the register window matches the current block start
  int tau_lo, tau_hi;   // smallest / largest lag of the task
  if (dense) {
    tau_lo = tk.tau0;
    tau_hi = tk.tau0 + cnt - 1;
  } else if (cnt == 0) {  // I sums only
    tau_lo = tau_hi = 0;
  } else {
    tau_lo = lags[tk.l0];
    tau_hi = lags[tk.l0 + cnt - 1];
#pragma unroll
    for (int i = 0; i < G; ++i)
      if (i < cnt && lane == 0) s_lags[warp * G + i] = lags[tk.l0 + i];  // read back by this warp only
  }
  __syncwarp();
  // batch-relative step from which every lag (j_all) / any lag (j_any) of the task has a frame pair
  const int j_all = (int)min((int64_t)1 << 30, max((int64_t)0, (int64_t)tau_hi - t0));
  const int j_any = (int)min((int64_t)1 << 30, max((int64_t)0, (int64_t)tau_lo - t0));
  const f2x* oldl = OLD + lane;

  int st = 0, slot0 = 0;  // slot0: ring slot of the current item's OLD chunk 0
  unsigned ph = 0;
  for (int item = 0; PERS || item == 0; ++item) {
  int tile = (int)(blockIdx.x / ngroups);
  bool waited = false;  // PERS: the barrier of the item's first step has been passed already
  if constexpr (PERS) {
    mbar_wait(&full[st], ph);  // first step of the next item
    tile = s_tile[st];
    if (tile < 0) break;
    waited = true;
  }
  const int64_t p = (int64_t)tile * kTilePx + lane;
  // per-item state: OLD rows of the item's first step
  const int base_row = slot0 * kChunk + offbase;
  wvalid = false;
  if (dense) {
    o0 = (base_row - tk.tau0) % DEPTH;
  } else {
#pragma unroll
    for (int i = 0; i < G; ++i)
      if (i < cnt) w[i] = (f2x)(unsigned)((base_row - s_lags[warp * G + i]) % DEPTH);
  }
  slot0 = (slot0 + V) % NSLOT;
  // prologue steps: the window is being filled, nothing to consume
#pragma unroll 1
  for (int j = 0; PERS && j < LEAD; ++j) {
    if (!waited) mbar_wait(&full[st], ph);
    waited = false;
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[st]);
    if (++st == stages) st = 0, ph ^= 1u;
  }
  for (int cseg = 0; cseg < nchunks; cseg += kFoldChunks) {  // fp32 partial sums span one segment of chunks
  const int cend = min(nchunks, cseg + kFoldChunks);
#pragma unroll 1
  for (int c = cseg; c < cend; ++c) {
    if (!waited) mbar_wait(&full[st], ph);
    waited = false;
    const f2x* newc = NEW + (size_t)st * kChunk * kRowF2 + lane;
    const int j0 = c * kChunk;
    if (j0 >= j_all && j0 + kChunk <= b) {
      // ---- fast chunk: every pair of every step exists ----
      if (doI) {
#pragma unroll 1
        for (int blk = 0; blk < kChunk / G; ++blk) {
#pragma unroll
          for (int u = 0; u < G; ++u) {
            const f2x zn = newc[(size_t)(blk * G + u) * kRowF2];
            i2 = fma2(zn, zn, i2);
            i1 = add2(i1, zn);
          }
        }
      }
      if (dense) {
        if (!wvalid) {  // (re)load the window: the G-1 OLD frames that precede the chunk's first one
#pragma unroll
          for (int q = 1; q < G; ++q) {
            int r = o0 - q;
            if (r < 0) r += DEPTH;
            w[G - q] = oldl[(size_t)r * kRowF2];
          }
          wvalid = true;
        }
        dense_chunk_dispatch(cnt, acc, w, newc, oldl, o0, DEPTH);
      } else {
        sparse_chunk_dispatch(cnt, acc, w, newc, oldl, DEPTH);
      }
    } else {
#pragma unroll 1
    for (int blk = 0; blk < kChunk / G; ++blk) {  // warm-up and the batch's last, partial chunk: checked per block
      const int jb = c * kChunk + blk * G;  // batch-relative index of the block's first step
      const int ns = min(G, b - jb);        // steps of this block inside the batch
      if (ns <= 0) break;
      const f2x* nb = newc + (size_t)blk * G * kRowF2;
      if (doI) {
#pragma unroll
        for (int u = 0; u < G; ++u) {
          if (u < ns) {
            const f2x zn = nb[(size_t)u * kRowF2];
            i2 = fma2(zn, zn, i2);
            i1 = add2(i1, zn);
          }
        }
      }
      if (jb + ns <= j_any) {
        wvalid = false;  // no pair of this task yet
      } else if (dense) {
        // ---- masked block: pair (step u, lag tau0 + g) exists iff u - g >= vbase, and u < ns.  All G lags of
        // the window are updated; the surplus ones of a short task are discarded at the fold. ----
        const int vbase = (int)max((int64_t)-64, (int64_t)tk.tau0 - t0 - jb);
        if (!wvalid) {  // (re)load the window; rows of frames before the first one are masked below
#pragma unroll
          for (int q = 1; q < G; ++q) {
            int r = o0 - q;
            if (r < 0) r += DEPTH;
            w[G - q] = oldl[(size_t)r * kRowF2];
          }
        }
        wvalid = ns == G;
        const f2x* ob = oldl + (size_t)o0 * kRowF2;
#pragma unroll
        for (int u = 0; u < G; ++u) {
          if (u < ns) {
            const f2x zn = nb[(size_t)u * kRowF2];
            w[u] = ob[(size_t)u * kRowF2];
#pragma unroll
            for (int g = 0; g < G; ++g)
              if (u - g >= vbase) upd2(acc[g], zn, w[(u - g + G) % G]);
          }
        }
      } else {
        // ---- masked block of a lag list: pair (step u, lag i) exists iff u >= u0_i, and u < ns ----
        sparse_masked_dispatch(cnt, ns, acc, w, nb, oldl, &s_lags[warp * G], t0 + jb);
      }
      if (dense) {
        o0 += G;
        if (o0 >= DEPTH) o0 -= DEPTH;
      } else {
#pragma unroll
        for (int i = 0; i < G; ++i) {
          if (i < cnt) {
            unsigned o = (unsigned)w[i] + G;
            if (o >= (unsigned)DEPTH) o -= DEPTH;
            w[i] = (f2x)o;
          }
        }
      }
    }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[st]);
    if (++st == stages) st = 0, ph ^= 1u;
  }
  // fold the fp32 partial sums (<= kFoldChunks * kChunk terms) into the fp64 totals: one reduction
  // (RED.ADD.F64 in L2, nothing returns to the SM) per (lag, pixel).  Every address has one writer per
  // launch, which folds in program order, and launches are stream ordered: the order of the additions
  // is fixed and the result deterministic.
#pragma unroll
  for (int g = 0; g < G; ++g) {
    if (g < cnt) atomicAdd(&totals[(int64_t)(tk.l0 + g) * P + p], (double)f2x_sum(acc[g]));
    acc[g] = 0ull;
  }
  if (doI) {
    atomicAdd(&I2[p], (double)f2x_sum(i2));
    atomicAdd(&I1[p].x, (double)__uint_as_float((unsigned)(i1 & 0xffffffffull)));
    atomicAdd(&I1[p].y, (double)__uint_as_float((unsigned)(i1 >> 32)));
    i2 = 0ull, i1 = 0ull;
  }
  }
  }
}

// ------------------------------------------------------------------------------------------------
// host: the lag plan.  Lags are cut into tasks (one consumer warp each) and tasks into groups (one CTA
// per group and pixel tile).  A run of >= kDenseMin consecutive lags becomes dense tasks of equal size
// <= kG; the other lags become sparse tasks.  A group takes consecutive lags while its consumer warps
// (<= kMaxTasks) and its shared-memory window (lag span) fit; the sparse lags of a group are then spread
// over the warps the dense tasks leave free, and tasks are placed on warps so that the four SM
// sub-partitions (warp id mod 4) carry equal FP32 work (longest-processing-time first).
// ------------------------------------------------------------------------------------------------
namespace {
struct Atom {
  int l0, cnt, kind;  // dense task, or one sparse lag (cnt = 1)
};

void close_group(const std::vector<int32_t>& L, const std::vector<Atom>& atoms, size_t a0, size_t a1, bool with_I,
                 std::vector<LagTask>& tasks, std::vector<LagGroup>& groups) {
  LagGroup g;
  g.task0 = (int)tasks.size();
  g.tau_min = L[atoms[a0].l0];
  g.tau_max = L[atoms[a1 - 1].l0 + atoms[a1 - 1].cnt - 1];
  int n_dense = 0, n_sparse = 0;
  for (size_t a = a0; a < a1; ++a) (atoms[a].kind == 0 ? n_dense : n_sparse) += 1;
  // sparse task size: small enough to use the free warps (up to 8 warps in all), large enough to fit them
  int s = 1;
  if (n_sparse > 0) {
    const int free_w = kMaxTasks - n_dense;
    const int want_w = std::max(1, std::min(free_w, 8 - std::min(n_dense, 7)));
    s = std::min(kSparseMax, std::max(1, (n_sparse + want_w - 1) / want_w));
    for (;; ++s) {  // stretches are cut separately: make sure the warps suffice
      int need = 0;
      size_t a = a0;
      while (a < a1) {
        if (atoms[a].kind == 0) { ++a; continue; }
        size_t e = a;
        while (e < a1 && atoms[e].kind == 1) ++e;
        need += ((int)(e - a) + s - 1) / s;
        a = e;
      }
      if (need <= free_w || s >= kSparseMax) break;
    }
  }
  size_t a = a0;
  while (a < a1) {
    if (atoms[a].kind == 0) {
      tasks.push_back(LagTask{L[atoms[a].l0], atoms[a].cnt, atoms[a].l0, 0});
      ++a;
      continue;
    }
    size_t e = a;
    while (e < a1 && atoms[e].kind == 1) ++e;
    const int n = (int)(e - a), nt = (n + s - 1) / s;
    int l = atoms[a].l0;
    for (int k = 0; k < nt; ++k) {  // equal sizes
      const int cnt = n / nt + (k < n % nt ? 1 : 0);
      tasks.push_back(LagTask{L[l], cnt, l, 1});
      l += cnt;
    }
    a = e;
  }
  g.ntasks = (int)tasks.size() - g.task0;
  g.flags = with_I ? 1 : 0;
  auto cost = [&](int k) {
    const LagTask& t = tasks[g.task0 + k];
    return ((t.kind & 1) == 0 ? 4 * t.cnt + 2 : 5 * t.cnt + 1) + ((t.kind & 2) ? 5 : 0);
  };
  if (with_I) {  // this group also accumulates the I sums (kind bit 1): on a warp of its own if one is free,
                 // else on its lightest task
    if (g.ntasks < kMaxTasks) {
      tasks.push_back(LagTask{0, 0, 0, 1 | 2});
      g.ntasks += 1;
    } else {
      int best = 0;
      for (int k = 1; k < g.ntasks; ++k)
        if (cost(k) < cost(best)) best = k;
      tasks[g.task0 + best].kind |= 2;
    }
  }
  // placement: heaviest task first onto the least loaded sub-partition that still has a free warp
  for (int w = 0; w < 16; ++w) g.warp_task[w] = -1;
  std::vector<int> order(g.ntasks);
  for (int k = 0; k < g.ntasks; ++k) order[k] = k;
  std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return cost(x) > cost(y); });
  int load[4] = {0, 0, 0, 0}, used[4] = {0, 0, 0, 0};
  for (int k : order) {
    int best = -1;
    for (int q = 0; q < 4; ++q)
      if (used[q] < kMaxTasks / 4 && (best < 0 || load[q] < load[best])) best = q;
    g.warp_task[used[best] * 4 + best] = (signed char)k;
    used[best] += 1;
    load[best] += cost(k);
  }
  groups.push_back(g);
}
}  // namespace

bool lag_plan(Ctx& c, int smem_sm, int cta_slots, int ntiles) {
  const std::vector<int32_t>& L = c.lags;
  // shared memory one CTA may use when kLagMinBlocks CTAs share an SM (1 KB per CTA is reserved)
  size_t budget = (size_t)std::max(0, smem_sm / kLagMinBlocks - 1024 - 512);  // 1 KB reserved + 512 B static per CTA
  budget = std::min(budget, (size_t)c.max_smem_optin);
  // atoms
  std::vector<Atom> atoms;
  for (int i = 0; i < c.n_lags;) {
    int j = i;
    while (j + 1 < c.n_lags && L[j + 1] == L[j] + 1) ++j;
    const int len = j - i + 1;
    if (len >= kDenseMin) {
      const int nt = (len + kG - 1) / kG;
      int l = i;
      for (int k = 0; k < nt; ++k) {
        const int cnt = len / nt + (k < len % nt ? 1 : 0);
        atoms.push_back(Atom{l, cnt, 0});
        l += cnt;
      }
    } else {
      for (int k = i; k <= j; ++k) atoms.push_back(Atom{k, 1, 1});
    }
    i = j + 1;
  }
  // greedy groups
  c.tasks.clear();
  c.groups.clear();
  auto fits = [&](size_t a0, size_t a1) {  // atoms [a0, a1) as one group
    const int tmin = L[atoms[a0].l0], tmax = L[atoms[a1 - 1].l0 + atoms[a1 - 1].cnt - 1];
    if (lag_smem_bytes(tmin, tmax, kMinStages + 1) > budget && a1 - a0 > 1) return false;
    int need = 0;
    size_t a = a0;
    while (a < a1) {
      if (atoms[a].kind == 0) { ++need; ++a; continue; }
      size_t e = a;
      while (e < a1 && atoms[e].kind == 1) ++e;
      need += ((int)(e - a) + kSparseMax - 1) / kSparseMax;
      a = e;
    }
    return need <= kMaxTasks;
  };
  std::vector<std::pair<size_t, size_t>> cuts;
  size_t a0 = 0;
  while (a0 < atoms.size()) {
    size_t a1 = a0 + 1;
    while (a1 < atoms.size() && fits(a0, a1 + 1)) ++a1;
    cuts.push_back({a0, a1});
    a0 = a1;
  }
  // the group with the fewest lags also accumulates the I sums of the batch
  size_t gI = 0;
  auto nl = [&](const std::pair<size_t, size_t>& r) {
    int n = 0;
    for (size_t a = r.first; a < r.second; ++a) n += atoms[a].cnt;
    return n;
  };
  for (size_t k = 1; k < cuts.size(); ++k)
    if (nl(cuts[k]) < nl(cuts[gI])) gI = k;
  for (size_t k = 0; k < cuts.size(); ++k) close_group(L, atoms, cuts[k].first, cuts[k].second, k == gI, c.tasks, c.groups);
  // pipeline depth: as deep as the widest group's window leaves room for
  int stages = kMaxStages;
  for (const LagGroup& g : c.groups)
    while (stages > kMinStages && lag_smem_bytes(g.tau_min, g.tau_max, stages) > budget) --stages;
  size_t smem = 0;
  for (const LagGroup& g : c.groups) smem = std::max(smem, lag_smem_bytes(g.tau_min, g.tau_max, stages));
  if (smem > (size_t)c.max_smem_optin) return false;  // a single task's own lag span does not fit
  c.lag_stages = stages;
  c.lag_smem = smem;
  // persistent CTAs: the cta_slots resident CTAs of the device are shared out in proportion to the groups' work
  // per pixel tile (FP32 work of the tasks + a constant for streaming the window), at least one CTA each
  {
    const int ng = (int)c.groups.size();
    std::vector<double> wgt(ng);
    double wsum = 0.0;
    for (int g = 0; g < ng; ++g) {
      double wg = 40.0;
      for (int k = 0; k < c.groups[g].ntasks; ++k) {
        const LagTask& t = c.tasks[c.groups[g].task0 + k];
        wg += ((t.kind & 1) == 0 ? 4.0 * t.cnt + 2.0 : 5.0 * t.cnt + 1.0) + ((t.kind & 2) ? 5.0 : 0.0);
      }
      wgt[g] = wg;
      wsum += wg;
    }
    const int slots = std::max(cta_slots, ng);
    int used = 0;
    for (int g = 0; g < ng; ++g) {
      int n = (int)(slots * wgt[g] / wsum);
      n = std::max(1, std::min(n, std::max(1, ntiles)));
      c.groups[g].nctas = n;
      used += n;
    }
    // hand the CTAs rounding left over to the heaviest groups
    for (int left = slots - used; left > 0;) {
      int best = -1;
      for (int g = 0; g < ng; ++g)
        if (c.groups[g].nctas < ntiles && (best < 0 || wgt[g] / c.groups[g].nctas > wgt[best] / c.groups[best].nctas)) best = g;
      if (best < 0) break;
      c.groups[best].nctas += 1;
      --left;
    }
    int at = 0;
    for (int g = 0; g < ng; ++g) {
      c.groups[g].cta0 = at;
      at += c.groups[g].nctas;
    }
    c.lag_grid = at;
  }
  return true;
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

// 2-D tensor map over the ring: dim0 = 2*P floats (32 pixels = 64 floats per box), dim1 = R ring slots
bool lag_make_tensor_map(Ctx& c) {
  typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                               const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
      qres != cudaDriverEntryPointSuccess)
    return false;
  const cuuint64_t gdim[2] = {(cuuint64_t)(2 * c.P), (cuuint64_t)c.R};
  const cuuint64_t gstride[1] = {(cuuint64_t)c.P * sizeof(float2)};
  const cuuint32_t box[2] = {(cuuint32_t)(2 * kTilePx), (cuuint32_t)kChunk};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = reinterpret_cast<EncodeFn>(fn)(&c.ring_map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, c.ring, gdim, gstride, box,
                                                    estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                                    CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

int launch_lag_tiled(Ctx& c, int64_t t0, int b) {
  cudaFuncSetAttribute(k_lag_tiled<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.lag_smem);
  cudaFuncSetAttribute(k_lag_tiled<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.lag_smem);
  cudaFuncSetAttribute(k_lag_tiled<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.lag_smem);
  cudaFuncSetAttribute(k_lag_tiled<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.lag_smem);
  const int ngroups = (int)c.groups.size();
  const int ntiles = (int)(c.P / kTilePx);
  // Persistent CTAs pay off where a CTA's fixed cost (launch, window fill, fold: ~8 us) outweighs its work: batches
  // of one or two chunks — provided the window prologue of a tile (LEAD steps) hides inside the pipeline depth and
  // the device is shared by at most two groups.  Measured on the B200 (profiles/r01_summary.md): lags 1..100,
  // batch 26: 35.8 -> 26.2 ms per 2000 frames; lags 1..208 (two groups): 66.5 -> 51.4 ms.  Elsewhere one CTA per
  // (tile, group) is as fast or faster: with a long window (isolated far lags) every tile costs LEAD barrier rounds
  // before its first chunk (lags 1..60 + 9 isolated lags <= 500, batch 26: 67 -> 147 ms); with many groups the
  // CTAs of a pixel tile launched side by side share the NEW frames in L2 and open the same DRAM pages (config 4:
  // 663 -> 852 ms); at long batches the fixed cost is amortised anyway (config 2: 13.95 -> 14.18 ms).
  int max_lead = 0;
  for (const LagGroup& g : c.groups) max_lead = std::max(max_lead, lag_lead(g.tau_min, g.tau_max));
  const bool persistent = c.lag_persistent >= 0 ? c.lag_persistent != 0
                                                : (b <= 2 * kChunk && ngroups <= 2 && max_lead <= c.lag_stages);
  const unsigned grid = persistent ? (unsigned)c.lag_grid : (unsigned)ntiles * (unsigned)ngroups;
  ProfScope ps(c, kKLag);
  // some group (other than the one that accumulates the I sums) has whole chunks without a pair in this batch
  bool skip = false;
  for (const LagGroup& g : c.groups) skip |= g.flags == 0 && (int64_t)g.tau_min - t0 >= kChunk && (int64_t)g.tau_min <= t0 + b - 1;
  auto kern = persistent ? (skip ? k_lag_tiled<true, true> : k_lag_tiled<true, false>)
                         : (skip ? k_lag_tiled<false, true> : k_lag_tiled<false, false>);
  if (persistent) cudaMemsetAsync(c.d_claim, 0, sizeof(int) * (size_t)ngroups, c.stream);
  kern<<<grid, (kMaxTasks + 1) * 32, c.lag_smem, c.stream>>>(c.ring_map, c.ring, c.R, c.P, t0, b, ngroups, c.lag_stages,
                                                              c.d_tasks, c.d_groups, c.d_lags, c.totals, c.I2, c.I1, ntiles,
                                                              c.d_claim);
  return 1;
}

}  // namespace nfs
