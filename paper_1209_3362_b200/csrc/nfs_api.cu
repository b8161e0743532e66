// nfs_api.cu — the C ABI of include/nfs.h: memory plan, host-side tables, stream orchestration.
// Every step of the hot path runs in the CUDA kernels of nfs_fft.cu / nfs_lag.cu / nfs_bin.cu;
// this file only plans, allocates, enqueues and copies results out.  No CPU fallback exists.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <memory>
#include <new>

#include "nfs_common.cuh"

using namespace nfs;

namespace {

bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }

// Every device buffer of a context comes from here.  With NFS_FLAG_GUARD each one sits between two guard zones of
// kGuardBytes filled with a canary byte, which nfs_check_guards reads back: an out-of-bounds write of any kernel next
// to one of the library's buffers is then detected (the substitute for compute-sanitizer memcheck where that tool is
// not available).
template <typename T>
bool dev_alloc(Ctx& c, T** p, size_t count) {
  void* q = nullptr;
  const size_t bytes = sizeof(T) * (count ? count : 1);
  const size_t user = (bytes + 255) / 256 * 256;
  const size_t g = c.guard ? kGuardBytes : 0;
  if (!cuda_ok(c, cudaMalloc(&q, user + 2 * g), "cudaMalloc")) return false;
  c.allocs.push_back(Ctx::Alloc{q, user});
  if (g && (!cuda_ok(c, cudaMemset(q, kGuardByte, g), "cudaMemset") ||
            !cuda_ok(c, cudaMemset(static_cast<char*>(q) + g + bytes, kGuardByte, (user - bytes) + g), "cudaMemset")))
    return false;
  *p = reinterpret_cast<T*>(static_cast<char*>(q) + g);
  c.dev_bytes += (int64_t)bytes;
  return true;
}

// |q| bins of the half plane (reading R6: b = floor(n_b |q| / q_Nyquist), uniform half-open bins on [0, pi) rad/px).
// A pixel with signed FFT-order indices (sx, sy) has (|q| / q_Nyquist)^2 = 4 (sx^2 H^2 + sy^2 W^2) / (W^2 H^2); it
// lies in bin b iff  b^2 W^2 H^2 <= 4 n_b^2 (sx^2 H^2 + sy^2 W^2) < (b + 1)^2 W^2 H^2.  The lower edges
// edge[b] = b^2 W^2 H^2 are tabulated once in 128-bit integers and a pixel's bin is found by bisection on them:
// exact, no division, no square root.
typedef unsigned __int128 u128;
struct BinEdges {
  std::vector<u128> edge;  // [n_b + 1]
  u128 scale;              // 4 n_b^2
  BinEdges(int W, int H, int nb) : edge((size_t)nb + 1), scale((u128)4 * (u128)nb * (u128)nb) {
    const u128 wh2 = (u128)((uint64_t)W * (uint64_t)W) * (u128)((uint64_t)H * (uint64_t)H);
    for (int b = 0; b <= nb; ++b) edge[(size_t)b] = (u128)((uint64_t)b * (uint64_t)b) * wh2;
  }
  // m = sx^2 H^2 + sy^2 W^2 (< 2^47 for frames up to 4096^2).  Returns -1 for the DC pixel and beyond the last edge.
  int bin_of(uint64_t m) const {
    if (m == 0) return -1;
    const u128 v = scale * (u128)m;
    if (v >= edge.back()) return -1;
    size_t lo = 0, hi = edge.size() - 1;  // invariant: edge[lo] <= v < edge[hi]
    while (hi - lo > 1) {
      const size_t mid = (lo + hi) / 2;
      (edge[mid] <= v ? lo : hi) = mid;
    }
    return (int)lo;
  }
};

// host tables: twiddles, bin map, lag plan
bool build_tables(Ctx& c) {
  const int W = c.W, H = c.H, n = c.n, nb = c.n_qbins;
  // twiddle tables of the FFT plan (nfs_fft.cu), evaluated in fp64 and rounded once.
  // L = W = H.  L <= 1024: one level, Li = L, Mi = L/32 lanes.  L > 1024: outer radix-32 pass over
  // T = L/32 threads, then inner FFTs of length Li = L/32 with Mi = Li/32 lanes.
  {
    const int L = W;
    const bool two = L > 1024;
    const int Li = two ? L / 32 : L, Mi = Li / 32;
    auto tw_of = [](int64_t num, int64_t den) {
      num %= den;
      // exact values on the axes and diagonals, fp64 elsewhere
      if (num == 0) return make_float2(1.f, 0.f);
      if (4 * num == den) return make_float2(0.f, -1.f);
      if (2 * num == den) return make_float2(-1.f, 0.f);
      if (4 * num == 3 * den) return make_float2(0.f, 1.f);
      const double ph = -2.0 * M_PI * (double)num / (double)den;
      return make_float2((float)cos(ph), (float)sin(ph));
    };
    std::vector<float2> tin((size_t)std::max(Li, 32));
    for (int j2 = 0; j2 < std::max(Mi, 1); ++j2)
      for (int k1 = 0; k1 < 32; ++k1) tin[(size_t)j2 * 32 + k1] = tw_of((int64_t)j2 * k1, Li);
    if (!dev_alloc(c, &c.tw, tin.size())) return false;
    if (!NFS_CUDA(c, cudaMemcpy(c.tw, tin.data(), sizeof(float2) * tin.size(), cudaMemcpyHostToDevice))) return false;
    if (two) {
      const int T = L / 32;
      std::vector<float2> tout((size_t)L);
      for (int k1 = 0; k1 < 32; ++k1)
        for (int j2 = 0; j2 < T; ++j2) tout[(size_t)k1 * T + j2] = tw_of((int64_t)j2 * k1, L);
      if (!dev_alloc(c, &c.tw_out, tout.size())) return false;
      if (!NFS_CUDA(c, cudaMemcpy(c.tw_out, tout.data(), sizeof(float2) * tout.size(), cudaMemcpyHostToDevice)))
        return false;
    }
  }

  // bin map in ring layout p = kx*H + ky: pixels grouped by bin in ascending p (fixed order, good locality), each
  // entry carrying its Hermitian weight: the columns 0 < kx < W/2 stand for two pixels of the full plane
  {
    const BinEdges edges(W, H, nb);
    const uint64_t H2 = (uint64_t)H * (uint64_t)H, W2 = (uint64_t)W * (uint64_t)W;
    std::vector<int32_t> binof((size_t)c.P);
    std::vector<int32_t> start((size_t)nb + 1, 0);
    c.counts.assign((size_t)nb, 0);
    for (int kx = 0; kx <= n; ++kx) {
      const uint64_t mx = (uint64_t)kx * (uint64_t)kx * H2;  // the Nyquist column kx = W/2 has |sx| = W/2
      for (int ky = 0; ky < H; ++ky) {
        const uint64_t ay = (uint64_t)std::min(ky, H - ky);  // |sy| of FFT-order index ky
        const int b = edges.bin_of(mx + ay * ay * W2);
        binof[(size_t)kx * H + ky] = b;
        if (b < 0) continue;
        start[(size_t)b + 1] += 1;
        c.counts[(size_t)b] += (kx == 0 || kx == n) ? 1 : 2;
      }
    }
    for (int b = 0; b < nb; ++b) start[(size_t)b + 1] += start[(size_t)b];
    std::vector<uint32_t> perm((size_t)start[(size_t)nb] ? (size_t)start[(size_t)nb] : 1);
    std::vector<int32_t> fill(start.begin(), start.end() - 1);
    for (int64_t p = 0; p < c.P; ++p) {
      const int b = binof[(size_t)p];
      if (b < 0) continue;
      const bool twice = p >= (int64_t)H && p < (int64_t)H * n;  // 0 < kx < n
      perm[(size_t)fill[(size_t)b]++] = (uint32_t)p | (twice ? 0x80000000u : 0u);
    }
    if (!dev_alloc(c, &c.perm, perm.size())) return false;
    if (!dev_alloc(c, &c.bin_start, (size_t)nb + 1)) return false;
    if (!NFS_CUDA(c, cudaMemcpy(c.perm, perm.data(), sizeof(uint32_t) * perm.size(), cudaMemcpyHostToDevice))) return false;
    if (!NFS_CUDA(c, cudaMemcpy(c.bin_start, start.data(), sizeof(int32_t) * ((size_t)nb + 1), cudaMemcpyHostToDevice)))
      return false;
  }

  // lag plan tables (nfs_lag.cu)
  if (!dev_alloc(c, &c.d_tasks, c.tasks.size())) return false;
  if (!dev_alloc(c, &c.d_groups, c.groups.size())) return false;
  if (!dev_alloc(c, &c.d_claim, c.groups.size())) return false;
  if (!dev_alloc(c, &c.d_lags, (size_t)c.n_lags)) return false;
  if (!NFS_CUDA(c, cudaMemcpy(c.d_tasks, c.tasks.data(), sizeof(LagTask) * c.tasks.size(), cudaMemcpyHostToDevice)))
    return false;
  if (!NFS_CUDA(c, cudaMemcpy(c.d_groups, c.groups.data(), sizeof(LagGroup) * c.groups.size(), cudaMemcpyHostToDevice)))
    return false;
  if (!NFS_CUDA(c, cudaMemcpy(c.d_lags, c.lags.data(), sizeof(int32_t) * c.n_lags, cudaMemcpyHostToDevice))) return false;
  return true;
}

void free_all(Ctx& c) {
  for (const Ctx::Alloc& a : c.allocs) cudaFree(a.base);
  c.allocs.clear();
  if (c.h_store) cudaFreeHost(c.h_store);
  c.h_store = nullptr;
  for (cudaEvent_t e : c.ev_pool) cudaEventDestroy(e);
  c.ev_pool.clear();
  if (c.own_stream && c.stream) cudaStreamDestroy(c.stream);
}

size_t totals_rows(const Ctx& c) { return (size_t)(c.bin_only ? c.max_group_lags : c.n_lags); }

bool zero_state(Ctx& c) {
  bool ok = true;
  ok &= NFS_CUDA(c, cudaMemsetAsync(c.totals, 0, sizeof(double) * totals_rows(c) * c.P, c.stream));
  if (c.bin_only)
    ok &= NFS_CUDA(c, cudaMemsetAsync(c.totals_b, 0, sizeof(double) * (size_t)c.n_lags * c.n_qbins, c.stream));
  ok &= NFS_CUDA(c, cudaMemsetAsync(c.I2, 0, sizeof(double) * (size_t)c.P, c.stream));
  ok &= NFS_CUDA(c, cudaMemsetAsync(c.I1, 0, sizeof(double2) * (size_t)c.P, c.stream));
  ok &= NFS_CUDA(c, cudaMemsetAsync(c.d_flags, 0, sizeof(int), c.stream));
  c.n_frames = 0;
  c.n_acc = 0;
  c.n_launches = 0;
  c.n_halo = 0;
  c.merged = false;
  c.merged_pairs.clear();
  c.merged_frames = 0;
  c.swept_frames = -1;
  c.ring_dirty = false;
  c.h2d_frames = c.d2h_frames = 0;
  return ok;
}

// synchronise and surface device-side flags
int sync_and_check(Ctx& c) {
  if (c.status != NFS_OK) return c.status;
  int flags = 0;
  if (!NFS_CUDA(c, cudaMemcpyAsync(&flags, c.d_flags, sizeof(int), cudaMemcpyDeviceToHost, c.stream))) return c.status;
  if (!NFS_CUDA(c, cudaStreamSynchronize(c.stream))) return c.status;
  if (flags & 1) c.status = NFS_ERR_ZERO_MEAN;
  return c.status;
}

// ring-layout double[P] ([kx][ky]) -> [H][W/2+1]
void ring_to_plane(const Ctx& c, const double* src, double* out) {
  const int n = c.n, H = c.H;
  for (int y = 0; y < H; ++y)
    for (int x = 0; x <= n; ++x) out[(size_t)y * (n + 1) + x] = src[(size_t)x * H + y];
}

// frames [f0, f1) between a ring of `slots` frames at `base` (slot = frame mod slots) and the pinned host store
bool copy_frames(Ctx& c, float2* base, int slots, int64_t f0, int64_t f1, bool to_device) {
  while (f0 < f1) {
    const int64_t s0 = f0 % slots;
    const int64_t n = std::min<int64_t>(f1 - f0, slots - s0);
    float2* dev = base + (size_t)s0 * c.P;
    float2* host = c.h_store + (size_t)f0 * c.P;
    const size_t bytes = sizeof(float2) * (size_t)n * c.P;
    if (!NFS_CUDA(c, to_device ? cudaMemcpyAsync(dev, host, bytes, cudaMemcpyHostToDevice, c.stream)
                               : cudaMemcpyAsync(host, dev, bytes, cudaMemcpyDeviceToHost, c.stream)))
      return false;
    (to_device ? c.h2d_frames : c.d2h_frames) += n;
    f0 += n;
  }
  return true;
}

// bring the totals of bands >= 1 up to date with the frames pushed so far (idempotent: they are rebuilt from zero)
bool run_band_sweeps(Ctx& c) {
  if (c.band_width <= 0 || c.n_bands <= 1 || c.swept_frames == c.n_frames) return true;
  const int l_first = c.band_l0[1];
  if (l_first < c.n_lags &&
      !NFS_CUDA(c, cudaMemsetAsync(c.totals + (size_t)l_first * c.P, 0, sizeof(double) * (size_t)(c.n_lags - l_first) * c.P, c.stream)))
    return false;
  c.ring_dirty = true;
  const bool ok = band_sweeps(
      c.n_frames, c.B, c.n_bands, c.band_l0, c.lags,
      [&](int64_t f0, int64_t f1) { return copy_frames(c, c.ring, c.R, f0, f1, true); },
      [&](int64_t f0, int64_t f1) { return copy_frames(c, c.ringN, c.RN, f0, f1, true); },
      [&](int64_t t0, int bb, int band) {
        c.n_launches += launch_lag_tiled(c, t0, bb, band);
        return NFS_CUDA(c, cudaGetLastError()) && c.status == NFS_OK;
      });
  if (ok) c.swept_frames = c.n_frames;
  return ok;
}

// step S5 (+ the I accumulators) for the frames transformed since the last accumulation
bool flush_pending(Ctx& c) {
  const int b = (int)(c.n_frames - c.n_acc);
  if (b <= 0) return true;
  c.n_launches += launch_lag_tiled(c, c.n_acc, b);
  if (!NFS_CUDA(c, cudaGetLastError())) return false;
  if (c.status != NFS_OK) return false;
  c.n_acc = c.n_frames;
  return true;
}

int create_impl(nfs_ctx** out, int W, int H, const int32_t* lags, int n_lags, int n_qbins, void* cuda_stream, int batch_frames,
                unsigned flags, int ring_frames_cap = 0, int64_t max_frames = 0) {
  if (!out) return NFS_ERR_INVALID_ARG;
  *out = nullptr;
  if (!lags_ok(lags, n_lags) || n_qbins < 1 || n_qbins > (1 << 20) || batch_frames < 0 || batch_frames > 8192)
    return NFS_ERR_INVALID_ARG;
  if ((flags & ~(unsigned)(NFS_FLAG_BIN_ONLY | NFS_FLAG_GUARD | NFS_FLAG_DIRECT)) != 0) return NFS_ERR_INVALID_ARG;
  if (!is_pow2(W) || !is_pow2(H) || W < 32 || H < 32 || W > 4096 || H > 4096) return NFS_ERR_INVALID_ARG;
  if (W != H) return NFS_ERR_UNSUPPORTED;
  if (n_lags > 65533) return NFS_ERR_INVALID_ARG;  // one grid row of the binning kernel per lag (+ I and V)

  // owned here until handed to the caller: every early return and a throwing host allocation (caught by NFS_GUARDED)
  // release the device memory, the stream and the context itself
  struct Release {
    void operator()(nfs_ctx* p) const {
      free_all(p->c);
      delete p;
    }
  };
  std::unique_ptr<nfs_ctx, Release> owner(new (std::nothrow) nfs_ctx());
  nfs_ctx* h = owner.get();
  if (!h) return NFS_ERR_OOM;
  Ctx& c = h->c;
  c.W = W;
  c.H = H;
  c.n = W / 2;
  c.P = (int64_t)H * (c.n + 1);
  c.n_lags = n_lags;
  c.n_qbins = n_qbins;
  c.lags.assign(lags, lags + n_lags);
  c.Lmax = lags[n_lags - 1];
  c.B = batch_frames > 0 ? batch_frames : 1024;
  c.R = c.Lmax + c.B;
  c.bin_only = (flags & NFS_FLAG_BIN_ONLY) != 0;
  c.guard = (flags & NFS_FLAG_GUARD) != 0;
  c.direct_only = (flags & NFS_FLAG_DIRECT) != 0;
  // band schedule: asked for by a ring capacity that cannot hold the whole lag window plus a batch
  if (ring_frames_cap < 0 || max_frames < 0) return NFS_ERR_INVALID_ARG;
  if (ring_frames_cap > 0 && ring_frames_cap < c.Lmax + (batch_frames > 0 ? batch_frames : 1)) {
    int b = 0, nstar = 0;
    if (c.bin_only) return NFS_ERR_UNSUPPORTED;  // band schedule with bin-only accumulation
    if (max_frames < 1 || !band_memory_plan(ring_frames_cap, batch_frames, &b, &nstar) || lags[0] > nstar)
      return NFS_ERR_INVALID_ARG;
    c.B = b;
    c.band_width = nstar;
    c.R = nstar + b;  // the FIFO of the paper: the OLD window of one band plus a batch
    c.RN = b;         // the "current image area"
    c.max_frames = max_frames;
  } else if (ring_frames_cap > 0 && batch_frames == 0) {
    c.B = std::max(1, std::min(1024, ring_frames_cap - c.Lmax));
    c.R = c.Lmax + c.B;
  }

  bool ok = NFS_CUDA(c, cudaGetDevice(&c.device));
  int smem_sm = 0;
  ok = ok && NFS_CUDA(c, cudaDeviceGetAttribute(&c.max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, c.device));
  ok = ok && NFS_CUDA(c, cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, c.device));
  ok = ok && NFS_CUDA(c, cudaDeviceGetAttribute(&c.n_sm, cudaDevAttrMultiProcessorCount, c.device));
  if (ok) {
    if (cuda_stream) {
      c.stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    } else {
      ok = NFS_CUDA(c, cudaStreamCreateWithFlags(&c.stream, cudaStreamNonBlocking));
      c.own_stream = ok;
    }
  }
  if (ok && !lag_plan(c, smem_sm, c.n_sm, c.P)) {
    c.status = NFS_ERR_INVALID_ARG;  // a lag task's own span does not fit shared memory
    ok = false;
  }
  if (ok) {
    // memory plan: everything is sized before the first frame arrives
    size_t free_b = 0, total_b = 0;
    ok = NFS_CUDA(c, cudaMemGetInfo(&free_b, &total_b));
    // default batch: 1024 frames, halved (down to 128) while the ring would take more than a third of the free memory
    while (ok && batch_frames == 0 && ring_frames_cap == 0 && c.B > 128 && (double)c.R * (double)c.P * 8.0 > (double)free_b / 3.0) {
      c.B /= 2;
      c.R = c.Lmax + c.B;
    }
    const double need = (double)c.P * ((double)(c.R + c.RN) * 8 + 8 + (double)totals_rows(c) * 8 + 8 + 16 + 8) +
                        (double)fft_rowT_elems(c) * 8 + (double)W * H * 4 + (double)(2 * n_lags + 2) * n_qbins * 8 +
                        (64 << 20);
    if (ok && need > (double)free_b) {
      c.status = NFS_ERR_OOM;
      ok = false;
    }
  }
  ok = ok && dev_alloc(c, &c.ring, (size_t)(c.R + c.RN) * c.P);
  if (ok && c.band_width > 0) {
    c.ringN = c.ring + (size_t)c.R * c.P;
    void* hp = nullptr;
    if (cudaHostAlloc(&hp, sizeof(float2) * (size_t)c.max_frames * c.P, cudaHostAllocDefault) != cudaSuccess) {
      cudaGetLastError();
      c.status = NFS_ERR_OOM;  // the pinned host store of the Fourier frames does not fit
      ok = false;
    }
    c.h_store = reinterpret_cast<float2*>(hp);
  }
  ok = ok && lag_configure(c);
  ok = ok && fft_configure(c);
  ok = ok && dev_alloc(c, &c.rowbuf, fft_rowT_elems(c));
  ok = ok && dev_alloc(c, &c.ref, (size_t)W * H);
  ok = ok && dev_alloc(c, &c.Fref, (size_t)c.P);
  ok = ok && dev_alloc(c, &c.totals, totals_rows(c) * c.P);
  if (c.bin_only) ok = ok && dev_alloc(c, &c.totals_b, (size_t)c.n_lags * c.n_qbins);
  ok = ok && dev_alloc(c, &c.I2, (size_t)c.P);
  ok = ok && dev_alloc(c, &c.I1, (size_t)c.P);
  ok = ok && dev_alloc(c, &c.sums, (size_t)c.B + 1);
  ok = ok && dev_alloc(c, &c.fft_cnt, fft_cnt_elems(c));
  ok = ok && dev_alloc(c, &c.d_out, (size_t)(c.n_lags + 2) * c.n_qbins);
  ok = ok && dev_alloc(c, &c.d_tmp, (size_t)c.P);
  ok = ok && dev_alloc(c, &c.d_flags, 1);
  ok = ok && dev_alloc(c, &c.d_npairs, (size_t)c.n_lags);
  ok = ok && dev_alloc(c, &c.d_fit, 4 * (size_t)c.n_qbins);
  ok = ok && build_tables(c);
  ok = ok && NFS_CUDA(c, cudaMemsetAsync(c.ring, 0, sizeof(float2) * (size_t)(c.R + c.RN) * c.P, c.stream));
  ok = ok && zero_state(c);
  ok = ok && NFS_CUDA(c, cudaStreamSynchronize(c.stream));
  if (ok) {
    *out = owner.release();
    return NFS_OK;
  }
  const int st = (c.status != NFS_OK) ? c.status : NFS_ERR_CUDA;
  const bool oom = c.cuda_err.find("out of memory") != std::string::npos;
  return oom ? NFS_ERR_OOM : st;  // `owner` frees everything
}

int get_plane(Ctx& c, double* out) {
  std::vector<double> tmp((size_t)c.P);
  if (!NFS_CUDA(c, cudaMemcpyAsync(tmp.data(), c.d_tmp, sizeof(double) * c.P, cudaMemcpyDeviceToHost, c.stream)))
    return c.status;
  const int st = sync_and_check(c);
  if (st != NFS_OK) return st;
  ring_to_plane(c, tmp.data(), out);
  return NFS_OK;
}

// common entry of the calls that read results: valid context, on its device, at least one frame, pairs up to date
int ready(nfs_ctx* h) {
  if (!h) return NFS_ERR_INVALID_ARG;
  Ctx& c = h->c;
  if (!enter(c)) return c.status;
  if (frames_in_I(c) < 1) return NFS_ERR_STATE;  // no frame yet, or only halo frames: every average would be 0 / 0
  if (!flush_pending(c)) return c.status;
  if (!run_band_sweeps(c)) return c.status;
  return NFS_OK;
}

}  // namespace

extern "C" {

int nfs_create_opts(nfs_ctx** out, int W, int H, const int32_t* lags, int n_lags, int n_qbins, void* cuda_stream,
                    int batch_frames, unsigned flags) {
  NFS_GUARDED(create_impl(out, W, H, lags, n_lags, n_qbins, cuda_stream, batch_frames, flags))
}

int nfs_create_banded(nfs_ctx** out, int W, int H, const int32_t* lags, int n_lags, int n_qbins, void* cuda_stream,
                      int batch_frames, unsigned flags, int ring_frames_cap, int64_t max_frames) {
  NFS_GUARDED(create_impl(out, W, H, lags, n_lags, n_qbins, cuda_stream, batch_frames, flags, ring_frames_cap, max_frames))
}

int nfs_get_transfer_counts(const nfs_ctx* h, int64_t* out) {
  if (!h || !out) return NFS_ERR_INVALID_ARG;
  const Ctx& c = h->c;
  out[0] = c.band_width > 0 ? c.n_bands : 1;
  out[1] = c.band_width;
  out[2] = c.h2d_frames;
  out[3] = c.d2h_frames;
  return NFS_OK;
}

int nfs_create_ex(nfs_ctx** out, int W, int H, const int32_t* lags, int n_lags, int n_qbins, void* cuda_stream,
                  int batch_frames) {
  return nfs_create_opts(out, W, H, lags, n_lags, n_qbins, cuda_stream, batch_frames, 0u);
}

int nfs_create(nfs_ctx** out, int W, int H, const int32_t* lags, int n_lags, int n_qbins, void* cuda_stream) {
  return nfs_create_opts(out, W, H, lags, n_lags, n_qbins, cuda_stream, 0, 0u);
}

static int push_impl(nfs_ctx* h, const uint16_t* d_frames, int n, bool halo) {
  if (!h || !d_frames || n < 1) return NFS_ERR_INVALID_ARG;
  if ((reinterpret_cast<uintptr_t>(d_frames) & 15u) != 0) return NFS_ERR_INVALID_ARG;  // 128-bit loads
  Ctx& c = h->c;
  if (!enter(c)) return c.status;
  if (c.merged) return NFS_ERR_STATE;  // the sums are those of all contexts: start over with nfs_reset
  if (halo && (c.n_frames != c.n_halo || c.band_width > 0 || c.n_frames + n > c.R - c.B)) return NFS_ERR_STATE;
  const int64_t fpx = (int64_t)c.W * c.H;
  if (c.band_width > 0) {
    if (c.n_frames + n > c.max_frames) return NFS_ERR_INVALID_ARG;  // the host store was sized for max_frames
    if (c.ring_dirty) {  // sweeps of an earlier finalize overwrote the streaming ring: bring its newest frames back
      if (!copy_frames(c, c.ring, c.R, std::max<int64_t>(0, c.n_frames - c.R), c.n_frames, true)) return c.status;
      c.ring_dirty = false;
    }
  }
  int done = 0;
  while (done < n) {
    // transform as many frames as the ring has room for; accumulate whenever a full batch is pending
    const int pending = (int)(c.n_frames - c.n_acc);
    const int b = std::min(c.B - pending, n - done);
    const uint16_t* fr = d_frames + (int64_t)done * fpx;
    if (c.n_frames == 0) c.n_launches += launch_make_ref(c, fr);
    c.n_launches += launch_fft_frames(c, fr, b, c.n_frames);
    if (c.status != NFS_OK) return c.status;
    // band schedule: every Fourier frame also goes to the pinned host store, once
    if (c.band_width > 0 && !copy_frames(c, c.ring, c.R, c.n_frames, c.n_frames + b, false)) return c.status;
    c.n_frames += b;
    done += b;
    if (halo) {  // halo frames only enter the ring: no pair has one of them as its later frame
      c.n_halo = c.n_frames;
      c.n_acc = c.n_frames;
    } else if (c.n_frames - c.n_acc == c.B && !flush_pending(c)) {
      return c.status;
    }
  }
  return NFS_OK;
}
int nfs_push_frames(nfs_ctx* h, const uint16_t* d_frames, int n) { NFS_GUARDED(push_impl(h, d_frames, n, false)) }
int nfs_push_halo(nfs_ctx* h, const uint16_t* d_frames, int n) { NFS_GUARDED(push_impl(h, d_frames, n, true)) }

// ---- partial sums of a context, for the one all-reduce of time-chunk sharding ----
// layout (doubles): [n_lags][P] pair sums (bin-only contexts: [n_lags][n_qbins]) | S2 [P] | S1 [P][2] | pairs [n_lags] | frames [1]
static int64_t partials_rows(const Ctx& c) { return c.bin_only ? (int64_t)c.n_qbins : c.P; }
int64_t nfs_partials_count(const nfs_ctx* h) {
  if (!h) return 0;
  const Ctx& c = h->c;
  return (int64_t)c.n_lags * partials_rows(c) + 3 * c.P + c.n_lags + 1;
}
static int export_impl(nfs_ctx* h, double* d_buf) {
  if (!h || !d_buf) return NFS_ERR_INVALID_ARG;
  Ctx& c = h->c;
  if (!enter(c)) return c.status;
  if (c.band_width > 0 || c.merged) return NFS_ERR_STATE;  // not combined with the band schedule; sums already replaced
  if (!flush_pending(c)) return c.status;
  const size_t nA = (size_t)c.n_lags * (size_t)partials_rows(c);
  const int64_t own = frames_in_I(c);
  if (own == 0) {
    // a rank whose time chunk is empty (more ranks than frames), or which has seen only halo frames, contributes
    // nothing: an all-zero buffer with frame count 0, so that it can still take part in the all-reduce
    if (!NFS_CUDA(c, cudaMemsetAsync(d_buf, 0, sizeof(double) * (size_t)nfs_partials_count(h), c.stream))) return c.status;
    return sync_and_check(c);
  }
  if (!NFS_CUDA(c, cudaMemcpyAsync(d_buf, c.bin_only ? c.totals_b : c.totals, sizeof(double) * nA, cudaMemcpyDeviceToDevice, c.stream)))
    return c.status;
  c.n_launches += launch_absolute_I(c, d_buf + nA, reinterpret_cast<double2*>(d_buf + nA + c.P));
  std::vector<double> tail((size_t)c.n_lags + 1);
  for (int l = 0; l < c.n_lags; ++l) tail[(size_t)l] = (double)pair_count(c, l);  // exact: counts < 2^53
  tail[(size_t)c.n_lags] = (double)own;
  if (!NFS_CUDA(c, cudaMemcpyAsync(d_buf + nA + 3 * c.P, tail.data(), sizeof(double) * tail.size(), cudaMemcpyHostToDevice, c.stream)))
    return c.status;
  return sync_and_check(c);
}
int nfs_export_partials(nfs_ctx* h, double* d_buf) { NFS_GUARDED(export_impl(h, d_buf)) }

static int import_impl(nfs_ctx* h, const double* d_buf) {
  if (!h || !d_buf) return NFS_ERR_INVALID_ARG;
  Ctx& c = h->c;
  if (!enter(c)) return c.status;
  // once per context (a second import would silently replace sums whose counts no longer describe the ring), and not
  // for the band schedule, whose bands >= 1 are rebuilt from the host store at every finalize
  // (a context without any frame may import: the rank of an empty time chunk receives the whole result like the others)
  if (c.merged || c.band_width > 0) return NFS_ERR_STATE;
  if (!flush_pending(c)) return c.status;
  const size_t nA = (size_t)c.n_lags * (size_t)partials_rows(c);
  std::vector<double> tail((size_t)c.n_lags + 1);
  bool ok = NFS_CUDA(c, cudaMemcpyAsync(c.bin_only ? c.totals_b : c.totals, d_buf, sizeof(double) * nA, cudaMemcpyDeviceToDevice, c.stream));
  ok = ok && NFS_CUDA(c, cudaMemcpyAsync(c.I2, d_buf + nA, sizeof(double) * (size_t)c.P, cudaMemcpyDeviceToDevice, c.stream));
  ok = ok && NFS_CUDA(c, cudaMemcpyAsync(c.I1, d_buf + nA + c.P, sizeof(double2) * (size_t)c.P, cudaMemcpyDeviceToDevice, c.stream));
  // the imported I sums are absolute: from here on the context's reference frame is zero
  ok = ok && NFS_CUDA(c, cudaMemsetAsync(c.Fref, 0, sizeof(float2) * (size_t)c.P, c.stream));
  ok = ok && NFS_CUDA(c, cudaMemcpyAsync(tail.data(), d_buf + nA + 3 * c.P, sizeof(double) * tail.size(), cudaMemcpyDeviceToHost, c.stream));
  if (!ok) return c.status;
  const int st = sync_and_check(c);
  if (st != NFS_OK) return st;
  c.merged_pairs.resize((size_t)c.n_lags);
  for (int l = 0; l < c.n_lags; ++l) c.merged_pairs[(size_t)l] = (int64_t)llround(tail[(size_t)l]);
  c.merged_frames = (int64_t)llround(tail[(size_t)c.n_lags]);
  c.merged = true;
  c.swept_frames = c.n_frames;
  return c.merged_frames >= 1 ? NFS_OK : NFS_ERR_STATE;
}
int nfs_import_partials(nfs_ctx* h, const double* d_buf) { NFS_GUARDED(import_impl(h, d_buf)) }

static int finalize_impl(nfs_ctx* h, double* D_q_tau, double* I_q, int64_t* counts) {
  const int rc = ready(h);
  if (rc != NFS_OK) return rc;
  Ctx& c = h->c;
  c.n_launches += launch_bin(c);
  if (c.status != NFS_OK) return c.status;
  const size_t nD = (size_t)c.n_lags * c.n_qbins;
  if (D_q_tau)
    if (!NFS_CUDA(c, cudaMemcpyAsync(D_q_tau, c.d_out, sizeof(double) * nD, cudaMemcpyDeviceToHost, c.stream)))
      return c.status;
  if (I_q)
    if (!NFS_CUDA(c, cudaMemcpyAsync(I_q, c.d_out + nD, sizeof(double) * c.n_qbins, cudaMemcpyDeviceToHost, c.stream)))
      return c.status;
  const int st = sync_and_check(c);
  if (st != NFS_OK) return st;
  if (counts) memcpy(counts, c.counts.data(), sizeof(int64_t) * c.n_qbins);
  return NFS_OK;
}
int nfs_finalize(nfs_ctx* h, double* D, double* I_q, int64_t* counts) { NFS_GUARDED(finalize_impl(h, D, I_q, counts)) }

int nfs_get_pair_counts(nfs_ctx* h, int64_t* n_pairs) {
  if (!h || !n_pairs) return NFS_ERR_INVALID_ARG;
  const Ctx& c = h->c;
  if (c.status != NFS_OK) return c.status;
  for (int l = 0; l < c.n_lags; ++l) n_pairs[l] = pair_count(c, l);
  return NFS_OK;
}

static int D2d_impl(nfs_ctx* h, int lag_index, double* out) {
  if (!h || !out) return NFS_ERR_INVALID_ARG;
  if (lag_index < 0 || lag_index >= h->c.n_lags) return NFS_ERR_INVALID_ARG;
  if (h->c.bin_only) return NFS_ERR_STATE;  // the 2-D difference spectra are not kept in this mode
  const int rc = ready(h);
  if (rc != NFS_OK) return rc;
  Ctx& c = h->c;
  c.n_launches += launch_D2d(c, lag_index, c.d_tmp);
  if (c.status != NFS_OK) return c.status;
  return get_plane(c, out);
}
int nfs_get_D2d(nfs_ctx* h, int lag_index, double* out) { NFS_GUARDED(D2d_impl(h, lag_index, out)) }

static int plane_impl(nfs_ctx* h, double* out, int which) {
  if (!h || !out) return NFS_ERR_INVALID_ARG;
  const int rc = ready(h);
  if (rc != NFS_OK) return rc;
  Ctx& c = h->c;
  c.n_launches += which == 0 ? launch_I2d(c, c.d_tmp) : launch_V2d(c, c.d_tmp);
  if (c.status != NFS_OK) return c.status;
  return get_plane(c, out);
}
int nfs_get_I2d(nfs_ctx* h, double* out) { NFS_GUARDED(plane_impl(h, out, 0)) }
int nfs_get_V2d(nfs_ctx* h, double* out) { NFS_GUARDED(plane_impl(h, out, 1)) }

static int variance_impl(nfs_ctx* h, double* V_q) {
  if (!V_q) return NFS_ERR_INVALID_ARG;
  const int rc = ready(h);
  if (rc != NFS_OK) return rc;
  Ctx& c = h->c;
  c.n_launches += launch_bin(c);
  if (c.status != NFS_OK) return c.status;
  if (!NFS_CUDA(c, cudaMemcpyAsync(V_q, c.d_out + (size_t)(c.n_lags + 1) * c.n_qbins, sizeof(double) * c.n_qbins,
                                   cudaMemcpyDeviceToHost, c.stream)))
    return c.status;
  return sync_and_check(c);
}
int nfs_get_variance(nfs_ctx* h, double* V_q) { NFS_GUARDED(variance_impl(h, V_q)) }

static int fit_impl(nfs_ctx* h, double* A_q, double* C_q, double* Gamma_q, double* chi2_q) {
  const int rc = ready(h);
  if (rc != NFS_OK) return rc;
  Ctx& c = h->c;
  c.n_launches += launch_bin(c);
  c.n_launches += launch_fit_eq1(c);
  if (c.status != NFS_OK) return c.status;
  double* dst[4] = {A_q, C_q, Gamma_q, chi2_q};
  for (int k = 0; k < 4; ++k)
    if (dst[k] && !NFS_CUDA(c, cudaMemcpyAsync(dst[k], c.d_fit + (size_t)k * c.n_qbins, sizeof(double) * c.n_qbins,
                                               cudaMemcpyDeviceToHost, c.stream)))
      return c.status;
  return sync_and_check(c);
}
int nfs_fit_eq1(nfs_ctx* h, double* A_q, double* C_q, double* Gamma_q, double* chi2_q) {
  NFS_GUARDED(fit_impl(h, A_q, C_q, Gamma_q, chi2_q))
}

int64_t nfs_num_frames(const nfs_ctx* h) { return h ? h->c.n_frames : 0; }
int nfs_ring_capacity(const nfs_ctx* h) { return h ? h->c.R : 0; }
int64_t nfs_device_bytes(const nfs_ctx* h) { return h ? h->c.dev_bytes : 0; }

int nfs_reset(nfs_ctx* h) {
  if (!h) return NFS_ERR_INVALID_ARG;
  Ctx& c = h->c;
  cudaStreamSynchronize(c.stream);
  cudaGetLastError();
  if (c.status == NFS_ERR_ZERO_MEAN) c.status = NFS_OK;
  if (!enter(c)) return c.status;  // a CUDA error is not recoverable by reset
  if (!zero_state(c)) return c.status;
  if (!NFS_CUDA(c, cudaStreamSynchronize(c.stream))) return c.status;
  return NFS_OK;
}

void nfs_destroy(nfs_ctx* h) {
  if (!h) return;
  cudaStreamSynchronize(h->c.stream);
  free_all(h->c);
  delete h;
}

const char* nfs_strerror(int status) {
  switch (status) {
    case NFS_OK: return "ok";
    case NFS_ERR_INVALID_ARG: return "invalid argument";
    case NFS_ERR_OOM: return "ring buffer and accumulators do not fit the free device memory";
    case NFS_ERR_CUDA: return "CUDA error (see nfs_last_cuda_error)";
    case NFS_ERR_ZERO_MEAN: return "a pushed frame summed to zero: normalisation by the spatial mean is undefined";
    case NFS_ERR_STATE: return "call not valid in this state";
    case NFS_ERR_UNSUPPORTED: return "unsupported configuration (W != H, or the band schedule together with NFS_FLAG_BIN_ONLY)";
    case NFS_ERR_TOO_LARGE: return "n_qbins exceeds NFS_STATIC_MAX_QBINS, the fixed scratch of nfs_azimuthal_mean_static";
    default: return "unknown status";
  }
}

const char* nfs_last_cuda_error(const nfs_ctx* h) { return h ? h->c.cuda_err.c_str() : ""; }

}  // extern "C"
