// nfs_probe.cu — measurement aid for bench.py (not on the hot path): the memory traffic of one small-batch launch of
// the lag-accumulation kernel (step S5) WITHOUT its arithmetic.  Same access pattern as k_lag_tiled in
// its HBM-bound regime: per pixel tile the window of LEAD + nchunks chunks is brought into shared memory by 2-D TMA
// boxes (tile pixels x kChunk ring slots, mbarrier pipeline), and every (lag, pixel) of the fp64 totals receives the
// RED.ADD.F64 the kernel issues per launch (one for a batch of one chunk, two for longer batches: opening and fold of a
// segment; the value added is 0.0, so the totals are left as they are).  What this kernel reaches is the ceiling
// of the pattern on this device; k_lag_tiled's distance to it is what its arithmetic, folds and bookkeeping cost.
#include "nfs_common.cuh"

namespace nfs {
namespace {

__device__ __forceinline__ unsigned p_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void p_mbar_init(uint64_t* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(p_smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void p_mbar_expect(uint64_t* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(p_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void p_mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(p_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void p_mbar_wait(uint64_t* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "PW_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra PD_%=;\n"
      "bra PW_%=;\n"
      "PD_%=:\n"
      "}\n" ::"r"(p_smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void p_tma_box(void* dst, const CUtensorMap* tmap, int c0, int c1, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n" ::"r"(
          p_smem_u32(dst)),
      "l"(tmap), "r"(c0), "r"(c1), "r"(p_smem_u32(bar))
      : "memory");
}

constexpr int kProbeStages = 8;
constexpr int kProbeWarps = 8;  // consumer warps; warp kProbeWarps issues the copies

// persistent CTAs; CTA i takes the tiles i, i + gridDim.x, ...  V chunks per tile starting at ring slot s_first.
template <int TPX>
__global__ void __launch_bounds__((kProbeWarps + 1) * 32) k_lag_probe(const __grid_constant__ CUtensorMap tmap, int V, int s_first,
                                                                      int ntiles, int n_lags, int n_red, int64_t P,
                                                                      double* __restrict__ totals) {
  extern __shared__ __align__(1024) unsigned char smraw[];
  uint64_t* full = reinterpret_cast<uint64_t*>(smraw);
  uint64_t* empty = full + kProbeStages;
  unsigned char* rows = smraw + 128;
  constexpr unsigned kBox = TPX * 8u * kChunk;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < kProbeStages; ++s) p_mbar_init(&full[s], 1), p_mbar_init(&empty[s], kProbeWarps);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();
  if (warp == kProbeWarps) {
    if (lane != 0) return;
    int st = 0;
    unsigned ph = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
      for (int m = 0; m < V; ++m) {
        p_mbar_wait(&empty[st], ph ^ 1u);
        p_tma_box(rows + (size_t)st * kBox, &tmap, 2 * tile * TPX, s_first + m * kChunk, &full[st]);
        p_mbar_expect(&full[st], kBox);
        if (++st == kProbeStages) st = 0, ph ^= 1u;
      }
    }
    return;
  }
  int st = 0;
  unsigned ph = 0;
  float sink = 0.f;
  for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    for (int m = 0; m < V; ++m) {
      p_mbar_wait(&full[st], ph);
      sink += reinterpret_cast<const float*>(rows + (size_t)st * kBox)[threadIdx.x];  // the chunk is touched once
      __syncwarp();
      if (lane == 0) p_mbar_arrive(&empty[st]);
      if (++st == kProbeStages) st = 0, ph ^= 1u;
    }
    // the totals of the tile: n_red reductions per (lag, pixel)
    for (int sub = 0; sub < TPX / 32; ++sub) {
      const int64_t p = (int64_t)tile * TPX + sub * 32 + lane;
      if (p < P)
        for (int l = warp; l < n_lags; l += kProbeWarps)
          for (int k = 0; k < n_red; ++k) atomicAdd(&totals[(int64_t)l * P + p], 0.0);
    }
  }
  if (sink == 123456.789f) totals[0] += 1.0;  // keeps the shared-memory reads alive
}

}  // namespace

// One launch of the probe for a batch of b frames; returns launches enqueued (1) and the algorithmic bytes it moves.
int launch_lag_probe(Ctx& c, int b, double* bytes) {
  const int tpx = c.lag_tpx;
  const int ntiles = (int)((c.P + tpx - 1) / tpx);
  const int lead = (c.Lmax + kChunk - 1) / kChunk, nchunks = (b + kChunk - 1) / kChunk;
  int V = lead + nchunks;
  if (V * kChunk > c.R) V = c.R / kChunk;
  const size_t smem = 128 + (size_t)kProbeStages * kChunk * tpx * 8;
  const int grid = std::min(ntiles, std::max(1, c.n_sm) * (tpx == 64 ? 2 : 4));
  const int n_red = b <= kChunk ? 1 : 2;
  if (bytes) *bytes = (double)c.P * (8.0 * V * kChunk + 16.0 * c.n_lags);
  if (tpx == 64) {
    if (!NFS_CUDA(c, cudaFuncSetAttribute(k_lag_probe<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem))) return 0;
    k_lag_probe<64><<<grid, (kProbeWarps + 1) * 32, smem, c.stream>>>(c.ring_map, V, 0, ntiles, c.n_lags, n_red, c.P, c.totals);
  } else {
    if (!NFS_CUDA(c, cudaFuncSetAttribute(k_lag_probe<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem))) return 0;
    k_lag_probe<32><<<grid, (kProbeWarps + 1) * 32, smem, c.stream>>>(c.ring_map, V, 0, ntiles, c.n_lags, n_red, c.P, c.totals);
  }
  NFS_CUDA(c, cudaGetLastError());
  return 1;
}

}  // namespace nfs
