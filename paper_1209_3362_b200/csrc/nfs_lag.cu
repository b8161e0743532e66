// nfs_lag.cu — step S5 of the hot path: lag accumulation  A_tau(p) += |F'_{s-tau}(p) - F'_s(p)|^2
// for every new frame s of a batch and every requested lag tau ("only the square
// moduli of FFT differences are evaluated N(N-1)/2 times"; L25 average over the measurement time).
//
// k_lag_tiled<NCW>: a CTA works on a tile of 4*NCW consecutive Fourier pixels (32 or 64) and one group of lags at
// a time.  A producer warp streams the batch through shared memory with TMA tensor copies (cp.async.bulk.tensor +
// mbarrier) into a ring of chunks that holds the lag window; the batch's own frames are the head of that ring
// (single stream) or, for a group whose smallest lag is far away, a second stream.  A consumer warp owns 32 pixels
// and one lag task:
//   * a run of consecutive lags tau0 .. tau0+cnt-1 (cnt <= 13): the smallest lag is accumulated directly
//     (|z_s - z_{s-tau0}|^2: sub.f32x2 + fma.rn.f32x2), every further lag through the difference of neighbouring lags
//        |z_s - z_{o-1}|^2 - |z_s - z_o|^2 = |z_{o-1}|^2 - |z_o|^2 - 2 Re( conj(z_s) (z_{o-1} - z_o) ),   o = s - tau,
//     i.e. ONE packed FMA per pair update on a rotating register window of the increments e_o = z_{o-1} - z_o; the
//     |z|^2 terms telescope to two boundary values per lag and fold interval.  This halves the arithmetic of the
//     dominant loop and, unlike the plain cross-term form, does not cancel in fp32: the
//     accumulated quantity is the small difference between neighbouring lags itself;
//   * a list of isolated lags (<= 6): one LDS.64 and the direct update per pair.
// fp32 partial sums are folded into the fp64 totals every kFoldChunks chunks and at the end of a tile
// (BASELINE.json north_star (4)).  One warp of the lightest group also adds the batch to the I sums (sum |F'|^2,
// sum F').  Two launch shapes (template parameter PERS, chosen per batch by launch_lag_tiled): one CTA per (pixel
// tile, lag group), or persistent CTAs that claim the pixel tiles of their group and keep the pipeline full across
// tiles.  Results do not depend on the shape or on the tile width.
#include <algorithm>

#include "nfs_common.cuh"

namespace nfs {

// ------------------------------------------------------------------------------------------------
// Warp-specialised kernel.  Warps 0..NCW-1 = consumers (warp w: task slot w & 7, 32-pixel sub-tile w >> 3; the plan
// places tasks on slots so that the four SM sub-partitions carry equal work), the last warp = producer (highest
// warp id: first in the issue arbiter, so loads are never starved by the math warps).
// Time is cut into chunks of kChunk = 2*kG steps.  Shared memory, in rows of TPX pixels (8 B each):
//   OLD  [(NSLOT + 1) * kChunk]  ring of NSLOT = LEAD + stages chunk slots; OLD row e holds frame
//                                E0 + e, E0 = t0 - tau_lo - LEAD*kChunk, at row e % (NSLOT*kChunk); the
//                                last kChunk rows duplicate slot 0 so that up to kChunk consecutive rows never wrap.
//                                tau_lo = 0 for a single-stream group (the batch's frames are "lag 0" of the window),
//                                else the group's smallest lag; LEAD = window span in chunks
//   NEW  [stages * kChunk]       two-stream groups only: the batch's own frames, chunk c in stage c % stages
// full[stage]: the producer's arrival + the bytes of its copies for one pipeline step; empty[stage]: the
// consumer warps.  One tile per CTA: step = consumer chunk c (OLD chunk c + LEAD, NEW chunk c; chunk 0 also
// brings OLD chunks 0..LEAD-1).  Persistent: every tile has LEAD prologue steps that bring one OLD chunk each,
// then one step per chunk (OLD chunk j, NEW chunk j - LEAD); steps and ring slots are numbered through all the
// tiles of the CTA, so the next tile's window streams in while the last chunks of the current one are consumed.
// A chunk of frames that is contiguous in the HBM ring is one 2-D TMA box (TPX pixels x kChunk ring slots); a chunk
// that straddles the ring's wrap-around or starts before the first frame falls back to one bulk copy per row.
// ------------------------------------------------------------------------------------------------
__host__ __device__ inline int lag_lead(int tau_lo, int tau_max) { return (tau_max - tau_lo + kChunk - 1) / kChunk; }
__host__ __device__ inline int lag_tau_lo(const LagGroup& g) { return (g.flags & 2) ? 0 : g.tau_min; }

static size_t lag_smem_bytes(int tau_lo, int tau_max, bool single, int stages, int tpx) {
  const int nslot = lag_lead(tau_lo, tau_max) + stages;
  return 128 + sizeof(float2) * (size_t)tpx * (size_t)((nslot + 1) * kChunk + (single ? 0 : stages * kChunk));
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
// producer side: wait with a suspend-time hint, so that the idle warp does not burn issue slots
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
      "r"(parity), "r"(20000u)
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
// 2-D tensor copy global -> shared (SASS UTMALDG): box = TPX pixels (2 TPX floats) x kChunk ring slots
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
__device__ __forceinline__ float f2x_lo(f2x v) { return __uint_as_float((unsigned)(v & 0xffffffffull)); }
__device__ __forceinline__ float f2x_hi(f2x v) { return __uint_as_float((unsigned)(v >> 32)); }
__device__ __forceinline__ float f2x_sum(f2x v) { return f2x_lo(v) + f2x_hi(v); }
__device__ __forceinline__ double norm2_f64(float2 z) { return (double)z.x * (double)z.x + (double)z.y * (double)z.y; }

// producer: bring frames f0 .. f0+kChunk-1 of this pixel tile into shared rows dst (and dup, if given).
// Returns the bytes this lane's copies will complete on the barrier.
template <int TPX>
__device__ __forceinline__ unsigned load_chunk(const CUtensorMap* tmap, const float2* __restrict__ ring, int R, int64_t P,
                                               int64_t p0, int64_t f0, f2x* dst, f2x* dup, uint64_t* bar, int lane) {
  constexpr unsigned kRowBytes = TPX * 8u;
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
      bulk_g2s(dst + (size_t)lane * TPX, src, kRowBytes, bar);
      bytes = kRowBytes;
      if (dup) {
        bulk_g2s(dup + (size_t)lane * TPX, src, kRowBytes, bar);
        bytes += kRowBytes;
      }
    }
  }
  return bytes;
}

// ---- register-window task with exactly CNT lags: one whole chunk in which every pair of every step exists ----
// acc[0]: direct sum of the smallest lag; acc[g], g >= 1: cross sum X_{g-1} = sum_s Re(conj(z_s) e_{s - tau0 - (g-1)});
// w: the 13 most recent increments e_o = z_{o-1} - z_o of the OLD stream o = s - tau0; zprev = z_{o-1}.
// Per step: 2 LDS.64 (issued one step ahead), the increment, the direct update (2) and CNT - 1 packed FMAs.  The
// chunk's kChunk OLD rows are contiguous (the ring's slot 0 is duplicated behind its last slot).
template <int CNT, int TPX>
__device__ __forceinline__ void dense_chunk(f2x (&acc)[kG], f2x (&w)[kG], f2x& zprev, bool& wvalid, const f2x* newc,
                                            const f2x* oldl, int& o0, int DEPTH) {
  if (!wvalid) {  // (re)build the window: the increments of the CNT-2 OLD frames that precede the chunk's first one
    int r = o0 - (CNT - 1);
    if (r < 0) r += DEPTH;
    f2x zz = oldl[(size_t)r * TPX];
#pragma unroll
    for (int k = CNT - 2; k >= 1; --k) {
      if (++r == DEPTH) r = 0;
      const f2x zk = oldl[(size_t)r * TPX];
      w[kG - k] = sub2(zz, zk);
      zz = zk;
    }
    zprev = zz;  // z of the OLD frame just before the chunk's first one
    wvalid = true;
  }
  const f2x* ob = oldl + (size_t)o0 * TPX;
  f2x zn = newc[0], zo = ob[0];
#pragma unroll
  for (int u = 0; u < kChunk; ++u) {
    f2x zn1 = zn, zo1 = zo;
    if (u + 1 < kChunk) {  // next step's operands: in flight while this step's FMAs issue
      zn1 = newc[(size_t)(u + 1) * TPX];
      zo1 = ob[(size_t)(u + 1) * TPX];
    }
    w[u % kG] = sub2(zprev, zo);
    zprev = zo;
    upd2(acc[0], zn, zo);
#pragma unroll
    for (int g = 1; g < CNT; ++g) acc[g] = fma2(zn, w[(u - (g - 1) + kChunk) % kG], acc[g]);
    zn = zn1;
    zo = zo1;
  }
  o0 += kChunk;
  if (o0 >= DEPTH) o0 -= DEPTH;
}
// One block of <= kG steps of a register-window task in which every pair of every step exists, but the batch may
// end inside it (ns <= kG steps): the same arithmetic as dense_chunk, one predicate per step.
template <int CNT, int TPX>
__device__ __forceinline__ void dense_block_partial(int ns, f2x (&acc)[kG], f2x (&w)[kG], f2x& zprev, bool& wvalid,
                                                    const f2x* nb, const f2x* oldl, int o0, int DEPTH) {
  if (!wvalid) {
    int r = o0 - (CNT - 1);
    if (r < 0) r += DEPTH;
    f2x zz = oldl[(size_t)r * TPX];
#pragma unroll
    for (int k = CNT - 2; k >= 1; --k) {
      if (++r == DEPTH) r = 0;
      const f2x zk = oldl[(size_t)r * TPX];
      w[kG - k] = sub2(zz, zk);
      zz = zk;
    }
    zprev = zz;
  }
  const f2x* ob = oldl + (size_t)o0 * TPX;
#pragma unroll
  for (int u = 0; u < kG; ++u) {
    if (u < ns) {
      const f2x zn = nb[(size_t)u * TPX], zo = ob[(size_t)u * TPX];
      w[u] = sub2(zprev, zo);
      zprev = zo;
      upd2(acc[0], zn, zo);
#pragma unroll
      for (int g = 1; g < CNT; ++g) acc[g] = fma2(zn, w[(u - (g - 1) + kG) % kG], acc[g]);
    }
  }
  wvalid = ns == kG;  // a shorter block ends the batch
}

// warp-uniform dispatch on the number of lags: the plan makes runs of kDenseMin..kG lags, mostly of kG and kG - 1
template <int TPX, int CNT = kG>
__device__ __forceinline__ void dense_chunk_dispatch(int cnt, f2x (&acc)[kG], f2x (&w)[kG], f2x& zprev, bool& wvalid,
                                                     const f2x* newc, const f2x* oldl, int& o0, int DEPTH) {
  if constexpr (CNT <= kDenseMin) {
    dense_chunk<kDenseMin, TPX>(acc, w, zprev, wvalid, newc, oldl, o0, DEPTH);
  } else {
    if (cnt == CNT)
      dense_chunk<CNT, TPX>(acc, w, zprev, wvalid, newc, oldl, o0, DEPTH);
    else
      dense_chunk_dispatch<TPX, CNT - 1>(cnt, acc, w, zprev, wvalid, newc, oldl, o0, DEPTH);
  }
}
template <int TPX, int CNT = kG>
__device__ __forceinline__ void dense_partial_dispatch(int cnt, int ns, f2x (&acc)[kG], f2x (&w)[kG], f2x& zprev,
                                                       bool& wvalid, const f2x* nb, const f2x* oldl, int o0, int DEPTH) {
  if constexpr (CNT <= kDenseMin) {
    dense_block_partial<kDenseMin, TPX>(ns, acc, w, zprev, wvalid, nb, oldl, o0, DEPTH);
  } else {
    if (cnt == CNT)
      dense_block_partial<CNT, TPX>(ns, acc, w, zprev, wvalid, nb, oldl, o0, DEPTH);
    else
      dense_partial_dispatch<TPX, CNT - 1>(cnt, ns, acc, w, zprev, wvalid, nb, oldl, o0, DEPTH);
  }
}
// ---- lag-list task with exactly CNT lags, whole chunk: the low word of w[i] holds the OLD row of lag i; its
// kChunk rows are contiguous (duplicated slot 0) ----
template <int CNT, int TPX>
__device__ __forceinline__ void sparse_chunk(f2x (&acc)[kG], f2x (&w)[kG], const f2x* newc, const f2x* oldl, int DEPTH) {
  const f2x* ol[CNT];
#pragma unroll
  for (int i = 0; i < CNT; ++i) ol[i] = oldl + (size_t)(unsigned)w[i] * TPX;
#pragma unroll
  for (int u = 0; u < kChunk; ++u) {
    const f2x zn = newc[(size_t)u * TPX];
#pragma unroll
    for (int i = 0; i < CNT; ++i) upd2(acc[i], zn, ol[i][(size_t)u * TPX]);
  }
#pragma unroll
  for (int i = 0; i < CNT; ++i) {
    unsigned o = (unsigned)w[i] + kChunk;
    if (o >= (unsigned)DEPTH) o -= DEPTH;
    w[i] = (f2x)o;
  }
}
template <int TPX>
__device__ __forceinline__ void sparse_chunk_dispatch(int cnt, f2x (&acc)[kG], f2x (&w)[kG], const f2x* newc, const f2x* oldl,
                                                      int DEPTH) {
  switch (cnt) {
    case 0: break;  // a task that only accumulates the I sums
    case 1: sparse_chunk<1, TPX>(acc, w, newc, oldl, DEPTH); break;
    case 2: sparse_chunk<2, TPX>(acc, w, newc, oldl, DEPTH); break;
    case 3: sparse_chunk<3, TPX>(acc, w, newc, oldl, DEPTH); break;
    case 4: sparse_chunk<4, TPX>(acc, w, newc, oldl, DEPTH); break;
    case 5: sparse_chunk<5, TPX>(acc, w, newc, oldl, DEPTH); break;
    default: sparse_chunk<kSparseMax, TPX>(acc, w, newc, oldl, DEPTH); break;  // lag lists of <= kSparseMax
  }
}

// the I sums of one chunk (sum |F'_s|^2, sum F'_s over the batch's frames): ns <= kChunk steps of the NEW rows,
// re-read from shared memory by the one warp of the group that carries them (outside the lag loops)
template <int TPX>
__device__ __forceinline__ void accumulate_I(const f2x* newc, int ns, int doI, f2x& i2, f2x& i1) {
  if (ns == kChunk) {
#pragma unroll
    for (int u = 0; u < kChunk; ++u) {
      const f2x zn = newc[(size_t)u * TPX];
      if (doI & 1) i2 = fma2(zn, zn, i2);
      if (doI & 2) i1 = add2(i1, zn);
    }
  } else {
#pragma unroll 1
    for (int u = 0; u < ns; ++u) {
      const f2x zn = newc[(size_t)u * TPX];
      if (doI & 1) i2 = fma2(zn, zn, i2);
      if (doI & 2) i1 = add2(i1, zn);
    }
  }
}

// One block of a lag-list task with exactly CNT lags in which some pairs do not exist (warm-up: the OLD
// frame would precede the first frame; or the batch's ragged tail): pair (step u, lag i) is counted iff
// u >= u0_i = lag_i - (frame number of step 0), and u < ns.
template <int CNT, int TPX>
__device__ __forceinline__ void sparse_masked(int ns, f2x (&acc)[kG], const f2x (&w)[kG], const f2x* nb, const f2x* oldl,
                                              const int* my_lags, int64_t frame0) {
  int u0[CNT];
#pragma unroll
  for (int i = 0; i < CNT; ++i) u0[i] = (int)min((int64_t)99, max((int64_t)0, (int64_t)my_lags[i] - frame0));
#pragma unroll
  for (int u = 0; u < kG; ++u) {
    if (u < ns) {
      const f2x zn = nb[(size_t)u * TPX];
#pragma unroll
      for (int i = 0; i < CNT; ++i)
        if (u >= u0[i]) upd2(acc[i], zn, oldl[(size_t)((unsigned)w[i] + u) * TPX]);
    }
  }
}
template <int TPX>
__device__ __forceinline__ void sparse_masked_dispatch(int cnt, int ns, f2x (&acc)[kG], const f2x (&w)[kG], const f2x* nb,
                                                       const f2x* oldl, const int* my_lags, int64_t frame0) {
  switch (cnt) {
    case 0: break;
    case 1: sparse_masked<1, TPX>(ns, acc, w, nb, oldl, my_lags, frame0); break;
    case 2: sparse_masked<2, TPX>(ns, acc, w, nb, oldl, my_lags, frame0); break;
    case 3: sparse_masked<3, TPX>(ns, acc, w, nb, oldl, my_lags, frame0); break;
    case 4: sparse_masked<4, TPX>(ns, acc, w, nb, oldl, my_lags, frame0); break;
    case 5: sparse_masked<5, TPX>(ns, acc, w, nb, oldl, my_lags, frame0); break;
    default: sparse_masked<kSparseMax, TPX>(ns, acc, w, nb, oldl, my_lags, frame0); break;
  }
}

// Fold of a register-window task after whole chunks: S(tau0) directly; S(tau + 1) = S(tau) - 2 X + |z_{sa - tau - 1}|^2
// - |z_{sb - tau}|^2 over the steps sa..sb of the whole chunks since the segment opened.  The first |z|^2 went into
// the totals when the segment opened, the second is the OLD row oend - g of the step after the last whole chunk (that
// chunk's window is still resident: call before the chunk that follows is released), everything in fp64.
template <int TPX>
__device__ __forceinline__ void dense_fold(f2x (&acc)[kG], int cnt, const f2x* oldl, int oend, int oopen, int DEPTH,
                                           double* tot, int64_t P, int64_t p) {
  double run = (double)f2x_sum(acc[0]);
  atomicAdd(&tot[p], run);
  int r = oend, r2 = oopen;
#pragma unroll
  for (int g = 1; g < kG; ++g) {
    if (g < cnt) {
      if (--r < 0) r += DEPTH;
      const f2x z = oldl[(size_t)r * TPX];
      run -= 2.0 * (double)f2x_sum(acc[g]) + norm2_f64(make_float2(f2x_lo(z), f2x_hi(z)));
      if (oopen >= 0) {  // one-chunk segment: the opening terms |z_{oopen - g}|^2 are still resident and join here (one
                         // reduction per lag and pixel instead of two)
        if (--r2 < 0) r2 += DEPTH;
        const f2x y = oldl[(size_t)r2 * TPX];
        run += norm2_f64(make_float2(f2x_lo(y), f2x_hi(y)));
      }
      atomicAdd(&tot[(int64_t)g * P + p], run);
    }
  }
#pragma unroll
  for (int g = 0; g < kG; ++g) acc[g] = 0ull;
}

template <int NCW, int SLOTS, bool PERS, bool SKIP>
__global__ void __launch_bounds__((NCW + 4) * 32, NCW <= 8 ? 2 : 1)
    k_lag_tiled(const __grid_constant__ CUtensorMap tmap, const float2* __restrict__ ring, int R,
                const __grid_constant__ CUtensorMap tmapN, const float2* __restrict__ ringN, int RN, int64_t P,
                int64_t t0_batch, int b_batch, int gbase, int ngroups, int lbase, int stages,
                const LagTask* __restrict__ tasks, const LagGroup* __restrict__ groups, const int32_t* __restrict__ lags,
                double* __restrict__ totals, double* __restrict__ I2, double2* __restrict__ I1, int ntiles,
                int* __restrict__ claim) {
  constexpr int G = kG;
  constexpr int TPX = 32 * (NCW / SLOTS);  // pixels per tile: one 32-pixel sub-tile per SLOTS consumer warps
  static_assert(NCW == SLOTS || NCW == 2 * SLOTS, "SLOTS task slots x 1 or 2 sub-tiles");
  static_assert(NCW + 4 <= 32, "at most 1024 threads");
  static_assert(kChunk % G == 0 && kChunk <= 32 && 2 * G - 1 <= kChunk, "a chunk is a whole number of G-step blocks, one lane per row");
  static_assert(kSparseMax == 6 && kSparseMax <= G, "sparse_chunk_dispatch lists cases 0..5 and the default");
  static_assert(SLOTS <= 16 && SLOTS % 4 == 0, "warp_task[16], whole sub-partition rounds");
  extern __shared__ __align__(128) unsigned char smraw[];
  __shared__ int s_lags[NCW * kG];  // the lags of each sparse task, for the warm-up path
  __shared__ int s_tile[kMaxStages];  // tile of the item whose first step uses this stage, or -1: no more work
  // persistent launch: group gi owns CTAs [cta0, cta0 + nctas), which claim the group's pixel tiles one after
  // the other (claim[gi], zeroed before the launch) and run through them without draining the shared-memory
  // pipeline.  One-tile launch: CTA = (tile, group), the groups of a tile side by side (they share L2 lines).
  int gi = gbase;
  if constexpr (PERS) {
    while (gi + 1 < gbase + ngroups && (int)blockIdx.x >= groups[gi].cta0 + groups[gi].nctas) ++gi;
  } else {
    gi = gbase + blockIdx.x % ngroups;
  }
  const LagGroup& grp = groups[gi];
  const int tau_min = grp.tau_min, tau_max = grp.tau_max;
  const bool withI = (grp.flags & 1) != 0;
  const bool single = (grp.flags & 2) != 0;
  // no frame pair of this group exists yet (the group that accumulates the I sums always runs)
  if (!withI && (int64_t)tau_min > t0_batch + b_batch - 1) return;
  // SKIP (launched only while some group's smallest lag still reaches back before frame 0): such a group skips
  // the whole chunks in which it has no pair, i.e. it works on the batch cut at the front (the I sums need every
  // frame: that group keeps the whole batch).  Otherwise t0 and b stay kernel parameters (no registers).
  int64_t t0 = t0_batch;
  int b = b_batch;
  if constexpr (SKIP) {
    if (!withI && (int64_t)tau_min > t0) {
      const int skip = (int)(((int64_t)tau_min - t0) / kChunk) * kChunk;
      t0 += skip;
      b -= skip;
    }
  }
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int tau_lo = single ? 0 : tau_min;
  const int LEAD = lag_lead(tau_lo, tau_max);
  const int NSLOT = LEAD + stages;
  const int DEPTH = NSLOT * kChunk;
  uint64_t* full = reinterpret_cast<uint64_t*>(smraw);      // [kMaxStages]
  uint64_t* empty = full + kMaxStages;                      // [kMaxStages]
  static_assert(2 * kMaxStages * 8 <= 128, "barriers fit the 128-byte header");
  f2x* OLD = reinterpret_cast<f2x*>(smraw + 128);           // [(NSLOT + 1) * kChunk][TPX]
  f2x* NEW = OLD + (size_t)(NSLOT + 1) * kChunk * TPX;      // [stages][kChunk][TPX], two-stream groups only
  const int nchunks = (b + kChunk - 1) / kChunk;
  // One item (pixel tile) = LEAD prologue steps that only bring OLD chunks (the window), then nchunks steps that
  // bring OLD chunk j (and NEW chunk j - LEAD) and are consumed.  Steps are numbered through all items of the
  // CTA: step v uses pipeline stage v % stages and puts its OLD chunk into ring slot v % NSLOT, which held the
  // OLD chunk of step v - NSLOT = v - LEAD - stages, last read by the consumers at step v - stages.
  const int V = nchunks + LEAD;

  if (tid == 0) {
    const unsigned nt = (unsigned)grp.ntasks * (NCW / SLOTS);
    for (int s = 0; s < stages; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], nt);
    }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();

  // Registers: the CTA is launched with a whole warpgroup for the producer (warps NCW..NCW+3, of which only the
  // first works), which gives its registers back (setmaxnreg.dec) so that the consumer warpgroups can grow theirs.
  if (warp >= NCW) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 24;\n");
    if (warp > NCW) return;
    // ------------------------------- producer -------------------------------
    const int64_t E0 = t0 - tau_lo - (int64_t)LEAD * kChunk;  // frame held by row 0 of an item's OLD chunk 0
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
        const int64_t p0 = (int64_t)tile * TPX;
        for (int j = 0; j < V; ++j) {
          mbar_wait_relaxed(&empty[st], ph ^ 1u);  // passes at once on the first use of a stage
          if (j == 0 && lane == 0) s_tile[st] = tile;  // ordered before the consumers' read by the arrive below
          f2x* dst = OLD + (size_t)slot * kChunk * TPX;
          f2x* dup = slot == 0 ? OLD + (size_t)NSLOT * kChunk * TPX : nullptr;
          unsigned bytes = load_chunk<TPX>(&tmap, ring, R, P, p0, E0 + (int64_t)j * kChunk, dst, dup, &full[st], lane);
          if (!single && j >= LEAD)
            bytes += load_chunk<TPX>(&tmapN, ringN, RN, P, p0, t0 + (int64_t)(j - LEAD) * kChunk,
                                     NEW + (size_t)st * kChunk * TPX, nullptr, &full[st], lane);
          bytes = __reduce_add_sync(0xffffffffu, bytes);
          if (lane == 0) mbar_arrive_expect_tx(&full[st], bytes);
          if (++st == stages) st = 0, ph ^= 1u;
          if (++slot == NSLOT) slot = 0;
        }
      }
    } else {
      // one pixel tile: the whole window (OLD chunks 0..LEAD) comes with the first chunk, no prologue steps
      const int64_t p0 = (int64_t)(blockIdx.x / ngroups) * TPX;
      for (int c = 0; c < nchunks; ++c) {
        if (c >= stages) mbar_wait_relaxed(&empty[st], ph ^ 1u);
        unsigned bytes = 0;
        if (!single)
          bytes = load_chunk<TPX>(&tmapN, ringN, RN, P, p0, t0 + (int64_t)c * kChunk, NEW + (size_t)st * kChunk * TPX, nullptr,
                                  &full[st], lane);
        for (int m = (c == 0 ? 0 : c + LEAD); m <= c + LEAD; ++m) {
          f2x* dst = OLD + (size_t)slot * kChunk * TPX;
          f2x* dup = slot == 0 ? OLD + (size_t)NSLOT * kChunk * TPX : nullptr;
          bytes += load_chunk<TPX>(&tmap, ring, R, P, p0, E0 + (int64_t)m * kChunk, dst, dup, &full[st], lane);
          if (++slot == NSLOT) slot = 0;
        }
        bytes = __reduce_add_sync(0xffffffffu, bytes);
        if (lane == 0) mbar_arrive_expect_tx(&full[st], bytes);
        if (++st == stages) st = 0, ph ^= 1u;
      }
    }
    return;
  }
  if constexpr (NCW <= 8)
    asm volatile("setmaxnreg.inc.sync.aligned.u32 104;\n");
  else
    asm volatile("setmaxnreg.inc.sync.aligned.u32 112;\n");

  // ------------------------------- consumers -------------------------------
  const int sub = warp / SLOTS;  // 32-pixel sub-tile of this warp
  const int tix = grp.warp_task[warp % SLOTS];
  if (tix < 0) return;
  const LagTask tk = tasks[grp.task0 + tix];
  const bool dense = (tk.kind & 1) == 0;
  const int doI = (tk.kind >> 1) & 3;  // bit 0: this warp also accumulates I2 += |F'_s|^2; bit 1: I1 += F'_s
  const int cnt = tk.cnt;
  f2x i2 = 0ull, i1 = 0ull;             // fp32 partials of the I sums (<= kFoldChunks * kChunk terms, like acc)
  // Dense task: acc[0] direct sum of lag tau0, acc[g] cross sum of lag tau0 + g against tau0 + g - 1; w = rotating
  // window of the G most recent increments of the OLD stream.  Sparse task: acc[i] direct sum of lag i; the low
  // word of w[i] holds the OLD row of lag i at the block start.
  f2x acc[G], w[G];
  f2x zprev = 0ull;
#pragma unroll
  for (int g = 0; g < G; ++g) acc[g] = 0ull, w[g] = 0ull;
  // OLD row (before the ring modulo) of the frame that lag tau pairs with step j:  j + offbase - tau
  const int offbase = LEAD * kChunk + tau_lo;
  int o0 = 0;           // dense: ring row of frame (t0 + jb - tau0) at the current block start
  bool wvalid = false;  // dense: the register window matches the current block start
  int tau_lo_t, tau_hi_t;  // smallest / largest lag of the task
  if (dense) {
    tau_lo_t = tk.tau0;
    tau_hi_t = tk.tau0 + cnt - 1;
  } else if (cnt == 0) {  // I sums only
    tau_lo_t = tau_hi_t = 0;
  } else {
    tau_lo_t = lags[tk.l0];
    tau_hi_t = lags[tk.l0 + cnt - 1];
#pragma unroll
    for (int i = 0; i < G; ++i)
      if (i < cnt && lane == 0) s_lags[warp * G + i] = lags[tk.l0 + i];  // read back by this warp only
  }
  __syncwarp();
  // batch-relative step from which every lag (j_all) / any lag (j_any) of the task has a frame pair
  const int j_all = (int)min((int64_t)1 << 30, max((int64_t)0, (int64_t)tau_hi_t - t0));
  const int j_any = (int)min((int64_t)1 << 30, max((int64_t)0, (int64_t)tau_lo_t - t0));
  const f2x* oldl = OLD + sub * 32 + lane;
  double* tot = totals + (int64_t)(tk.l0 - lbase) * P;  // row of the task's first lag

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
  const int64_t p = (int64_t)tile * TPX + sub * 32 + lane;
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
  int nslot = slot0 + LEAD;  // single stream: ring slot of the item's NEW chunk 0 (= OLD chunk LEAD)
  if (nslot >= NSLOT) nslot -= NSLOT;
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
  bool open = false;  // dense: whole chunks have been accumulated in this segment (their boundary terms are open)
  int oend = 0;       // dense: OLD row of the step after the segment's last whole chunk
  int oopen = -1;     // dense, one-chunk segment: OLD row at its opening (the opening terms are added at the fold)
#pragma unroll 1
  for (int c = cseg; c < cend; ++c) {
    if (!waited) mbar_wait(&full[st], ph);
    waited = false;
    const f2x* newc = (single ? OLD + (size_t)nslot * kChunk * TPX : NEW + (size_t)st * kChunk * TPX) + sub * 32 + lane;
    if (++nslot == NSLOT) nslot = 0;
    const int j0 = c * kChunk;
    if (doI) accumulate_I<TPX>(newc, min(kChunk, b - j0), doI, i2, i1);
    if (j0 >= j_all && j0 + kChunk <= b) {
      // ---- fast chunk: every pair of every step exists ----
      if (dense) {
        if (!open && cend - cseg == 1) {
          open = true;
          oopen = o0;  // the window of this one chunk is still resident at the fold
        }
        if (!open) {
          // first whole chunk of the segment: the |z|^2 of the OLD frames just before it enter the totals of the
          // further lags (they telescope against the ones subtracted at the fold): lag tau0 + g gets
          // sum_{k=1..g} |z_{o0-k}|^2, in fp64
          open = true;
          double pre = 0.0;
          int r = o0;
#pragma unroll
          for (int g = 1; g < G; ++g) {
            if (g < cnt) {
              if (--r < 0) r += DEPTH;
              const f2x z = oldl[(size_t)r * TPX];
              pre += norm2_f64(make_float2(f2x_lo(z), f2x_hi(z)));
              if (p < P) atomicAdd(&tot[(int64_t)g * P + p], pre);
            }
          }
        }
        dense_chunk_dispatch<TPX>(cnt, acc, w, zprev, wvalid, newc, oldl, o0, DEPTH);
        oend = o0;
      } else {
        sparse_chunk_dispatch<TPX>(cnt, acc, w, newc, oldl, DEPTH);
      }
    } else {
#pragma unroll 1
    for (int blk = 0; blk < kChunk / G; ++blk) {  // warm-up and the batch's last, partial chunk: checked per block
      const int jb = c * kChunk + blk * G;  // batch-relative index of the block's first step
      const int ns = min(G, b - jb);        // steps of this block inside the batch
      if (ns <= 0) break;
      const f2x* nb = newc + (size_t)blk * G * TPX;
      if (jb + ns <= j_any) {
        // no pair of this task yet
      } else if (dense && jb >= j_all) {
        // ---- the batch's last chunk: every pair of the block's ns steps exists: same recurrence, predicated steps ----
        if (!open) {
          open = true;
          double pre = 0.0;
          int r = o0;
#pragma unroll
          for (int g = 1; g < G; ++g) {
            if (g < cnt) {
              if (--r < 0) r += DEPTH;
              const f2x z = oldl[(size_t)r * TPX];
              pre += norm2_f64(make_float2(f2x_lo(z), f2x_hi(z)));
              if (p < P) atomicAdd(&tot[(int64_t)g * P + p], pre);
            }
          }
        }
        dense_partial_dispatch<TPX>(cnt, ns, acc, w, zprev, wvalid, nb, oldl, o0, DEPTH);
        oend = o0 + ns;
        if (oend >= DEPTH) oend -= DEPTH;
      } else if (dense) {
        // ---- masked block of a run of lags: every existing pair directly, pair (step u, lag tau0 + g) exists
        // iff u - g >= vbase and u < ns; straight into the fp64 totals (rare: the warm-up of a stack and the
        // ragged tail of a batch).  Rows o0 - (G-1) .. o0 + G-1 are contiguous thanks to the duplicated slot. ----
        if (open) {  // (not reached in practice: warm-up blocks precede the whole chunks) fold what is open first
          if (p < P) dense_fold<TPX>(acc, cnt, oldl, oend, oopen, DEPTH, tot, P, p);
          open = false;
          oopen = -1;
        }
        const int vbase = (int)max((int64_t)-64, (int64_t)tk.tau0 - t0 - jb);
        int rb = o0 - (G - 1);
        if (rb < 0) rb += DEPTH;
        const f2x* ob = oldl + (size_t)rb * TPX;
#pragma unroll
        for (int g = 0; g < G; ++g) {
          if (g < cnt) {
            f2x a = 0ull;
#pragma unroll 1
            for (int u = max(0, vbase + g); u < ns; ++u) upd2(a, nb[(size_t)u * TPX], ob[(size_t)(G - 1 + u - g) * TPX]);
            if (p < P) atomicAdd(&tot[(int64_t)g * P + p], (double)f2x_sum(a));
          }
        }
        wvalid = false;
      } else {
        // ---- masked block of a lag list: pair (step u, lag i) exists iff u >= u0_i, and u < ns ----
        sparse_masked_dispatch<TPX>(cnt, ns, acc, w, nb, oldl, &s_lags[warp * G], t0 + jb);
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
    if (c == cend - 1) break;  // the segment's last chunk is released after the fold below, which reads its window rows
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[st]);
    if (++st == stages) st = 0, ph ^= 1u;
  }
// fold the fp32 partial sums (<= kFoldChunks * kChunk terms) into the fp64 totals: one reduction
  // (RED.ADD.F64 in L2, nothing returns to the SM) per (lag, pixel).  Every address has one writer per
  // launch, which folds in program order, and launches are stream ordered: the order of the additions
  // is fixed and the result deterministic.
  if (p < P) {
    if (dense) {
      if (open) dense_fold<TPX>(acc, cnt, oldl, oend, oopen, DEPTH, tot, P, p);
    } else {
#pragma unroll
      for (int g = 0; g < G; ++g)
        if (g < cnt) atomicAdd(&tot[(int64_t)g * P + p], (double)f2x_sum(acc[g]));
    }
    if (doI & 1) atomicAdd(&I2[p], (double)f2x_sum(i2));
    if (doI & 2) {
      atomicAdd(&I1[p].x, (double)f2x_lo(i1));
      atomicAdd(&I1[p].y, (double)f2x_hi(i1));
    }
  }
#pragma unroll
  for (int g = 0; g < G; ++g) acc[g] = 0ull;
  i2 = 0ull, i1 = 0ull;
  __syncwarp();
  if (lane == 0) mbar_arrive(&empty[st]);
  if (++st == stages) st = 0, ph ^= 1u;
  }
  }
}

// ------------------------------------------------------------------------------------------------
// host: the lag plan.  Lags are cut into tasks (one consumer warp each per 32-pixel sub-tile) and tasks into groups
// (one CTA per group and pixel tile).  A run of >= kDenseMin consecutive lags becomes dense tasks of equal size
// <= kG; the other lags become sparse tasks.  A group takes consecutive lags while its task slots (<= kTaskSlots)
// and its shared-memory window (lag span) fit; the sparse lags of a group are then spread over the slots the dense
// tasks leave free, and tasks are placed on slots so that the four SM sub-partitions (warp id mod 4) carry equal
// FP32 work (longest-processing-time first).
// ------------------------------------------------------------------------------------------------
namespace {
struct Atom {
  int l0, cnt, kind;  // dense task, or one sparse lag (cnt = 1)
};

// issue slots per time step: a run costs 2 loads, the increment, the direct update (2) and one FMA per further lag;
// a lag list one load and two packed operations per lag plus the load of the new frame
double task_cost(const LagTask& t) {
  const double lag_cost = t.cnt == 0 ? 0.0 : ((t.kind & 1) == 0 ? 4.0 + t.cnt : 3.0 * t.cnt + 1.0);
  return lag_cost + ((t.kind & 6) ? 1.0 : 0.0) + ((t.kind & 2) ? 1.0 : 0.0) + ((t.kind & 4) ? 1.0 : 0.0);
}

void close_group(const std::vector<int32_t>& L, const std::vector<Atom>& atoms, size_t a0, size_t a1, bool with_I, int slots,
                 std::vector<LagTask>& tasks, std::vector<LagGroup>& groups) {
  LagGroup g;
  g.task0 = (int)tasks.size();
  g.tau_min = L[atoms[a0].l0];
  g.tau_max = L[atoms[a1 - 1].l0 + atoms[a1 - 1].cnt - 1];
  int n_dense = 0, n_sparse = 0;
  for (size_t a = a0; a < a1; ++a) (atoms[a].kind == 0 ? n_dense : n_sparse) += 1;
  // sparse task size: small enough to use the free slots, large enough to fit them
  int s = 1;
  if (n_sparse > 0) {
    const int free_w = slots - n_dense;
    s = std::min(kSparseMax, std::max(1, (n_sparse + free_w - 1) / std::max(1, free_w)));
    for (;; ++s) {  // stretches are cut separately: make sure the slots suffice
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
  if (with_I) {  // this group also accumulates the I sums (kind bits 1, 2): on a slot of its own if one is free,
                 // else on its lightest tasks
    if (g.ntasks < slots) {
      tasks.push_back(LagTask{0, 0, 0, 1 | 2 | 4});
      g.ntasks += 1;
    } else {
      // sum |F'|^2 (bit 1) and sum F' (bit 2) ride on the lightest task (the last one among equals): it re-reads the
      // chunk's NEW rows, three issue slots per step.  If that task is part of a run of consecutive lags it hands up
      // to three lags to the tasks before it in the run that have room, so that it stays no heavier than they are.
      int best = 0;
      for (int k = 1; k < g.ntasks; ++k)
        if (task_cost(tasks[g.task0 + k]) <= task_cost(tasks[g.task0 + best])) best = k;
      LagTask* T = &tasks[g.task0];
      T[best].kind |= 6;
      for (int moved = 0; moved < 3 && (T[best].kind & 1) == 0 && T[best].cnt > kDenseMin; ++moved) {
        int k = best;  // nearest earlier task of the same run with room
        while (k > 0 && (T[k - 1].kind & 1) == 0 && T[k - 1].tau0 + T[k - 1].cnt == T[k].tau0 && T[k - 1].cnt >= kG) --k;
        if (k == 0 || (T[k - 1].kind & 1) != 0 || T[k - 1].tau0 + T[k - 1].cnt != T[k].tau0) break;
        T[k - 1].cnt += 1;  // it takes the first lag of task k; every task from k to best - 1 shifts up by one lag
        for (int q = k; q < best; ++q) T[q].tau0 += 1, T[q].l0 += 1;
        T[best].tau0 += 1, T[best].l0 += 1, T[best].cnt -= 1;
      }
    }
  }
  // placement: heaviest task first onto the least loaded sub-partition that still has a free slot
  for (int w = 0; w < 16; ++w) g.warp_task[w] = -1;
  std::vector<int> order(g.ntasks);
  for (int k = 0; k < g.ntasks; ++k) order[k] = k;
  std::stable_sort(order.begin(), order.end(),
                   [&](int x, int y) { return task_cost(tasks[g.task0 + x]) > task_cost(tasks[g.task0 + y]); });
  double load[4] = {0, 0, 0, 0};
  int used[4] = {0, 0, 0, 0};
  for (int k : order) {
    int best = -1;
    for (int q = 0; q < 4; ++q)
      if (used[q] < slots / 4 && (best < 0 || load[q] < load[best])) best = q;
    g.warp_task[used[best] * 4 + best] = (signed char)k;
    used[best] += 1;
    load[best] += task_cost(tasks[g.task0 + k]);
  }
  g.cta0 = g.nctas = 0;
  groups.push_back(g);
}
}  // namespace

static bool plan_with(Ctx& c, int slots, int smem_sm, int n_sm, int64_t P, int dense_max = kG) {
  const std::vector<int32_t>& L = c.lags;
  // shared memory a CTA may use: the opt-in maximum (one CTA per SM) bounds a group's window; two CTAs of 32-pixel
  // tiles share an SM when the plan's footprint allows it (1 KB per CTA is reserved, 1 KB static)
  const size_t budget = (size_t)std::max(0, std::min(smem_sm - 2048, c.max_smem_optin - 1024));
  // band of a lag in the out-of-core schedule: lags (k N*, (k+1) N*] form band k; no task or group
  // straddles two bands, and only band 0 streams its batch as the head of its window
  auto band_of = [&](int tau) { return c.band_width > 0 ? (tau - 1) / c.band_width : 0; };
  // atoms
  std::vector<Atom> atoms;
  for (int i = 0; i < c.n_lags;) {
    int j = i;
    while (j + 1 < c.n_lags && L[j + 1] == L[j] + 1 && band_of(L[j + 1]) == band_of(L[i])) ++j;
    const int len = j - i + 1;
    if (len >= kDenseMin && !c.direct_only) {  // NFS_FLAG_DIRECT: every lag is summed by the plain difference form
      const int nt = (len + dense_max - 1) / dense_max;
      int l = i;
      for (int k = 0; k < nt; ++k) {
        const int cnt = len / nt + (k < len % nt ? 1 : 0);
        if (cnt >= kDenseMin) {
          atoms.push_back(Atom{l, cnt, 0});
        } else {
          for (int q = 0; q < cnt; ++q) atoms.push_back(Atom{l + q, 1, 1});
        }
        l += cnt;
      }
    } else {
      for (int k = i; k <= j; ++k) atoms.push_back(Atom{k, 1, 1});
    }
    i = j + 1;
  }
  // greedy groups: a group is streamed as a single window when that costs no more shared memory than two streams
  auto single_of = [&](int tmin, int tmax) {
    return band_of(tmin) == 0 && lag_smem_bytes(0, tmax, true, kMinStages, 32) <= lag_smem_bytes(tmin, tmax, false, kMinStages, 32);
  };
  c.tasks.clear();
  c.groups.clear();
  auto fits = [&](size_t a0, size_t a1) {  // atoms [a0, a1) as one group
    const int tmin = L[atoms[a0].l0], tmax = L[atoms[a1 - 1].l0 + atoms[a1 - 1].cnt - 1];
    if (band_of(tmin) != band_of(tmax)) return false;
    const bool sg = single_of(tmin, tmax);
    if (lag_smem_bytes(sg ? 0 : tmin, tmax, sg, kMinStages, 32) > budget && a1 - a0 > 1) return false;
    int need = 0;
    size_t a = a0;
    while (a < a1) {
      if (atoms[a].kind == 0) { ++need; ++a; continue; }
      size_t e = a;
      while (e < a1 && atoms[e].kind == 1) ++e;
      need += ((int)(e - a) + kSparseMax - 1) / kSparseMax;
      a = e;
    }
    return need <= slots;
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
  c.max_group_lags = 0;
  for (size_t k = 0; k < cuts.size(); ++k) {  // (band schedule: among the groups of band 0, which run as the frames stream in)
    if (band_of(L[atoms[cuts[k].first].l0]) == 0 && nl(cuts[k]) < nl(cuts[gI])) gI = k;
    c.max_group_lags = std::max(c.max_group_lags, nl(cuts[k]));
  }
  for (size_t k = 0; k < cuts.size(); ++k) close_group(L, atoms, cuts[k].first, cuts[k].second, k == gI, slots, c.tasks, c.groups);
  for (LagGroup& g : c.groups)
    if (single_of(g.tau_min, g.tau_max)) g.flags |= 2;
  c.n_bands = band_of(L.back()) + 1;
  c.band_g0.assign((size_t)c.n_bands + 1, (int)c.groups.size());
  c.band_l0.assign((size_t)c.n_bands + 1, c.n_lags);
  for (int g = (int)c.groups.size() - 1; g >= 0; --g)
    for (int k = 0; k <= band_of(c.groups[g].tau_min); ++k) c.band_g0[(size_t)k] = g;
  for (int l = c.n_lags - 1; l >= 0; --l)
    for (int k = 0; k <= band_of(L[l]); ++k) c.band_l0[(size_t)k] = l;
  // tile width and pipeline depth.  64-pixel tiles (16 consumer warps, one CTA per SM, 512-byte rows) when every
  // group's window then still leaves kMinStages + 1 stages; else 32-pixel tiles, two CTAs per SM if they fit.
  auto smem_for = [&](int stages, int tpx) {
    size_t m = 0;
    for (const LagGroup& g : c.groups) m = std::max(m, lag_smem_bytes(lag_tau_lo(g), g.tau_max, (g.flags & 2) != 0, stages, tpx));
    return m;
  };
  int tpx = 32, per_sm = 1, stages = kMinStages;
  if (slots == kTaskSlots && P % 64 == 0 && smem_for(kMinStages + 1, 64) <= budget) {
    tpx = 64;
    stages = kMinStages + 1;
    while (stages < kMaxStages && smem_for(stages + 1, 64) <= budget) ++stages;
  } else {
    const size_t half = (size_t)std::max(0, smem_sm / 2 - 2048);
    if (slots == kTaskSlots && smem_for(kMinStages + 1, 32) <= half) {
      per_sm = 2;
      stages = kMinStages + 1;
      while (stages < kMaxStages && smem_for(stages + 1, 32) <= half) ++stages;
    } else {
      while (stages < kMaxStages && smem_for(stages + 1, 32) <= budget) ++stages;
    }
  }
  const size_t smem = smem_for(stages, tpx);
  if (smem > (size_t)c.max_smem_optin) return false;  // a single task's own lag span does not fit
  c.lag_stages = stages;
  c.lag_smem = smem;
  c.lag_tpx = tpx;
  c.lag_slots = slots;
  c.lag_ctas_per_sm = per_sm;
  // persistent CTAs: the resident CTAs of the device are shared out in proportion to the groups' work per pixel
  // tile (issue slots of the tasks + a constant for streaming the window), at least one CTA each
  {
    const int ntiles = (int)std::min<int64_t>((P + tpx - 1) / tpx, 1 << 30);
    const int ng = (int)c.groups.size();
    std::vector<double> wgt(ng);
    double wsum = 0.0;
    for (int g = 0; g < ng; ++g) {
      double wg = 20.0;
      for (int k = 0; k < c.groups[g].ntasks; ++k) wg += task_cost(c.tasks[c.groups[g].task0 + k]);
      wgt[g] = wg;
      wsum += wg;
    }
    const int slots = std::max(per_sm * std::max(1, n_sm), ng);
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

// The plan nfs_create uses.  Eight task slots per group with 64-pixel tiles (16 consumer warps) or two CTAs of
// 32-pixel tiles per SM; a plan whose window leaves room for one 32-pixel CTA per SM only (long lag spans: isolated
// lags) is redone with sixteen task slots, so that sixteen consumer warps share the SM there too.
bool lag_plan(Ctx& c, int smem_sm, int n_sm, int64_t P) {
  if (!plan_with(c, kTaskSlots, smem_sm, n_sm, P)) return false;
  if (c.lag_tpx == 32 && c.lag_ctas_per_sm == 1) {
    Ctx alt = c;
    if (plan_with(alt, 2 * kTaskSlots, smem_sm, n_sm, P, kDenseMaxWide)) {
      c.tasks = alt.tasks, c.groups = alt.groups;
      c.lag_stages = alt.lag_stages, c.lag_smem = alt.lag_smem, c.lag_tpx = alt.lag_tpx, c.lag_slots = alt.lag_slots;
      c.lag_ctas_per_sm = alt.lag_ctas_per_sm, c.lag_grid = alt.lag_grid, c.max_group_lags = alt.max_group_lags;
      c.n_bands = alt.n_bands, c.band_g0 = alt.band_g0, c.band_l0 = alt.band_l0;
    }
  }
  return true;
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
namespace {
typedef void (*LagKernel)(const CUtensorMap, const float2*, int, const CUtensorMap, const float2*, int, int64_t, int64_t, int, int, int, int, int, const LagTask*,
                          const LagGroup*, const int32_t*, double*, double*, double2*, int, int*);
template <int NCW, int SLOTS>
LagKernel lag_kernel_of(bool pers, bool skip) {
  return pers ? (skip ? k_lag_tiled<NCW, SLOTS, true, true> : k_lag_tiled<NCW, SLOTS, true, false>)
              : (skip ? k_lag_tiled<NCW, SLOTS, false, true> : k_lag_tiled<NCW, SLOTS, false, false>);
}
// (tile pixels, task slots): (64, 8) 16 consumer warps on two sub-tiles; (32, 8) 8 consumer warps, two CTAs per SM
// where they fit; (32, 16) 16 consumer warps on sixteen tasks
LagKernel lag_kernel(int tpx, int slots, bool pers, bool skip) {
  if (slots == 2 * kTaskSlots) return lag_kernel_of<2 * kTaskSlots, 2 * kTaskSlots>(pers, skip);
  if (tpx == 64) return lag_kernel_of<2 * kTaskSlots, kTaskSlots>(pers, skip);
  return lag_kernel_of<kTaskSlots, kTaskSlots>(pers, skip);
}
}  // namespace

// once at create, after the ring is allocated: the 2-D tensor map over the ring (dim0 = 2*P floats, box of one pixel
// tile; dim1 = R ring slots, box of kChunk) and the dynamic shared memory of the four launch variants
bool lag_configure(Ctx& c) {
  typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                               const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (!NFS_CUDA(c, cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres))) return false;
  if (!fn || qres != cudaDriverEntryPointSuccess) {
    c.status = NFS_ERR_CUDA;
    c.cuda_err = "cuTensorMapEncodeTiled not available";
    return false;
  }
  const cuuint64_t gstride[1] = {(cuuint64_t)c.P * sizeof(float2)};
  const cuuint32_t box[2] = {(cuuint32_t)(2 * c.lag_tpx), (cuuint32_t)kChunk};
  const cuuint32_t estr[2] = {1, 1};
  for (int which = 0; which < (c.band_width > 0 ? 2 : 1); ++which) {  // the ring; band schedule: also the NEW ring of the sweeps
    const cuuint64_t gdim[2] = {(cuuint64_t)(2 * c.P), (cuuint64_t)(which ? c.RN : c.R)};
    const CUresult r = reinterpret_cast<EncodeFn>(fn)(which ? &c.ringN_map : &c.ring_map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2,
                                                      which ? c.ringN : c.ring, gdim, gstride, box, estr,
                                                      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                                      CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
      c.status = NFS_ERR_CUDA;
      c.cuda_err = "cuTensorMapEncodeTiled failed";
      return false;
    }
  }
  for (int v = 0; v < 4; ++v)
    if (!NFS_CUDA(c, cudaFuncSetAttribute(lag_kernel(c.lag_tpx, c.lag_slots, (v & 1) != 0, (v & 2) != 0),
                                          cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.lag_smem)))
      return false;
  return true;
}

int launch_lag_tiled(Ctx& c, int64_t t0, int b, int band) {
  // band schedule: only the groups of one band per launch; a sweep (band > 0) takes the batch's own
  // frames from the NEW ring, the streaming pass (band 0) from the ring itself
  const bool banded = c.band_width > 0;
  const int g0 = banded ? c.band_g0[(size_t)band] : 0;
  const int ngroups = banded ? c.band_g0[(size_t)band + 1] - g0 : (int)c.groups.size();
  if (ngroups <= 0) return 0;
  const bool sweep = banded && band > 0;
  const CUtensorMap& mapN = sweep ? c.ringN_map : c.ring_map;
  const float2* ringN = sweep ? c.ringN : c.ring;
  const int RN = sweep ? c.RN : c.R;
  const int tpx = c.lag_tpx;
  const int ntiles = (int)((c.P + tpx - 1) / tpx);
  const int nthreads = (c.lag_slots * (tpx / 32) + 4) * 32;
  int n = 0;
  if (c.bin_only) {
    // PAPER.md:L41 ("store the entire 2D power spectra, which might be unnecessary"): one lag group per launch into
    // a per-pixel scratch of that group's lags, reduced into the |q|-binned totals in a fixed order right after
    int lbase = 0;
    for (int g = 0; g < ngroups; ++g) {
      const LagGroup& grp = c.groups[g];
      int nl = 0;
      for (int k = 0; k < grp.ntasks; ++k) nl += c.tasks[grp.task0 + k].cnt;
      const bool runs = (grp.flags & 1) || (int64_t)grp.tau_min <= t0 + b - 1;
      if (runs) {
        const bool skip = !(grp.flags & 1) && (int64_t)grp.tau_min - t0 >= kChunk;
        {
          ProfScope ps(c, kKLag);
          if (!NFS_CUDA(c, cudaMemsetAsync(c.totals, 0, sizeof(double) * (size_t)nl * c.P, c.stream))) return n;
          lag_kernel(tpx, c.lag_slots, false, skip)<<<(unsigned)ntiles, nthreads, c.lag_smem, c.stream>>>(
              c.ring_map, c.ring, c.R, c.ring_map, c.ring, c.R, c.P, t0, b, g, 1, lbase, c.lag_stages, c.d_tasks, c.d_groups,
              c.d_lags, c.totals, c.I2, c.I1, ntiles, c.d_claim);
          n += 1;
        }
        n += launch_bin_accumulate(c, lbase, nl);
      }
      lbase += nl;
    }
    return n;
  }
  // Persistent CTAs pay off where a CTA's fixed cost (launch, window fill, fold) outweighs its work: batches of one
  // or two chunks — provided the window prologue of a tile (LEAD steps) hides inside the pipeline depth and the
  // device is shared by at most two groups.  Elsewhere one CTA per (tile, group) is as fast or faster: with a long
  // window every tile costs LEAD barrier rounds before its first chunk; with many groups the CTAs of a pixel tile
  // launched side by side share the batch's frames in L2 and open the same DRAM pages; at long batches the fixed
  // cost is amortised anyway (measurements: profiles/).
  int max_lead = 0;
  for (const LagGroup& g : c.groups) max_lead = std::max(max_lead, lag_lead(lag_tau_lo(g), g.tau_max));
  const bool persistent =
      !banded && (c.lag_shape ? c.lag_shape == 2 : (b <= 2 * kChunk && ngroups <= 2 && max_lead <= c.lag_stages));
  const unsigned grid = persistent ? (unsigned)c.lag_grid : (unsigned)ntiles * (unsigned)ngroups;
  ProfScope ps(c, kKLag);
  // some group (other than the one that accumulates the I sums) has whole chunks without a pair in this batch
  bool skip = false;
  for (int g = g0; g < g0 + ngroups; ++g)
    skip |= !(c.groups[g].flags & 1) && (int64_t)c.groups[g].tau_min - t0 >= kChunk && (int64_t)c.groups[g].tau_min <= t0 + b - 1;
  if (persistent && !NFS_CUDA(c, cudaMemsetAsync(c.d_claim, 0, sizeof(int) * (size_t)ngroups, c.stream))) return 0;
  lag_kernel(tpx, c.lag_slots, persistent, skip)<<<grid, nthreads, c.lag_smem, c.stream>>>(
      c.ring_map, c.ring, c.R, mapN, ringN, RN, c.P, t0, b, g0, ngroups, 0, c.lag_stages, c.d_tasks, c.d_groups, c.d_lags,
      c.totals, c.I2, c.I1, ntiles, c.d_claim);
  return 1;
}

}  // namespace nfs
