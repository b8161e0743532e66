// nfs_api.cu — the C ABI of include/nfs.h: memory plan, host-side tables, stream orchestration.
// Every step of the hot path runs in the CUDA kernels of nfs_fft.cu / nfs_lag.cu / nfs_bin.cu;
// this file only plans, allocates, enqueues and copies results out.  No CPU fallback exists.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <new>

#include "nfs_common.cuh"

using namespace nfs;

struct nfs_ctx {
  Ctx c;
};

namespace {

bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }

// record the first CUDA error (sticky)
bool cuda_ok(Ctx& c, cudaError_t e, const char* what) {
  if (e == cudaSuccess) return true;
  if (c.status == NFS_OK) {
    c.status = NFS_ERR_CUDA;
    c.cuda_err = std::string(what) + ": " + cudaGetErrorString(e);
  }
  return false;
}
#define NFS_CUDA(c, call) cuda_ok((c), (call), #call)

bool check_launch(Ctx& c, const char* what) { return cuda_ok(c, cudaGetLastError(), what); }

template <typename T>
bool dev_alloc(Ctx& c, T** p, size_t count) {
  void* q = nullptr;
  const size_t bytes = sizeof(T) * (count ? count : 1);
  if (!cuda_ok(c, cudaMalloc(&q, bytes), "cudaMalloc")) return false;
  *p = reinterpret_cast<T*>(q);
  c.dev_bytes += (int64_t)bytes;
  return true;
}

uint64_t isqrt_u64(uint64_t v) {
  uint64_t r = (uint64_t)sqrt((double)v);
  while (r * r > v) --r;
  while ((r + 1) * (r + 1) <= v) ++r;
  return r;
}

// |q| bin of half-plane pixel (kx in [0, W/2], ky in [0, H)) by exact integer arithmetic (reading R6):
// b = isqrt(floor(4 nb^2 (kx'^2 H^2 + ky'^2 W^2) / (W^2 H^2))); DC and b >= nb excluded (-1).
int qbin_of(int kx, int ky, int W, int H, int nb) {
  const int64_t sx = kx;  // kx <= W/2; the Nyquist index has |kx'| = W/2
  const int64_t sy = ky < H / 2 ? ky : ky - H;
  if (sx == 0 && sy == 0) return -1;
  const unsigned __int128 num = (unsigned __int128)(4ull * (uint64_t)nb * (uint64_t)nb) *
                                ((unsigned __int128)((uint64_t)(sx * sx) * (uint64_t)H * (uint64_t)H) +
                                 (unsigned __int128)((uint64_t)(sy * sy) * (uint64_t)W * (uint64_t)W));
  const unsigned __int128 den = (unsigned __int128)((uint64_t)W * (uint64_t)W) * ((uint64_t)H * (uint64_t)H);
  const uint64_t b = isqrt_u64((uint64_t)(num / den));
  return b >= (uint64_t)nb ? -1 : (int)b;
}

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

  // bin map in ring layout: p = kx*H + ky
  std::vector<int32_t> start(nb + 1, 0);
  c.counts.assign(nb, 0);
  std::vector<int32_t> binof((size_t)c.P);
  for (int ky = 0; ky < H; ++ky)
    for (int kx = 0; kx <= n; ++kx) {
      const int64_t p = (int64_t)kx * H + ky;
      const int b = qbin_of(kx, ky, W, H, nb);
      binof[p] = b;
      if (b >= 0) {
        start[b + 1] += 1;
        c.counts[b] += (kx == 0 || kx == n) ? 1 : 2;
      }
    }
  for (int b = 0; b < nb; ++b) start[b + 1] += start[b];
  std::vector<uint32_t> perm((size_t)start[nb] ? (size_t)start[nb] : 1);
  {
    std::vector<int32_t> fill(start.begin(), start.end() - 1);
    for (int64_t p = 0; p < c.P; ++p) {  // ascending p inside each bin: fixed order, good locality
      const int b = binof[p];
      if (b < 0) continue;
      const bool interior = p >= (int64_t)H && p < (int64_t)H * n;  // 0 < kx < n: Hermitian weight 2
      perm[fill[b]++] = (uint32_t)p | (interior ? 0x80000000u : 0u);
    }
  }
  if (!dev_alloc(c, &c.perm, perm.size())) return false;
  if (!dev_alloc(c, &c.bin_start, (size_t)nb + 1)) return false;
  if (!NFS_CUDA(c, cudaMemcpy(c.perm, perm.data(), sizeof(uint32_t) * perm.size(), cudaMemcpyHostToDevice))) return false;
  if (!NFS_CUDA(c, cudaMemcpy(c.bin_start, start.data(), sizeof(int32_t) * (nb + 1), cudaMemcpyHostToDevice)))
    return false;

  // lag plan (nfs_lag.cu): tasks per consumer warp, groups per CTA, pipeline depth
  const std::vector<int32_t>& L = c.lags;
  int dev = 0, smem_sm = 0, n_sm = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev);
  cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  if (!lag_plan(c, smem_sm, kLagMinBlocks * std::max(1, n_sm), (int)(c.P / kTilePx))) {
    c.status = NFS_ERR_INVALID_ARG;
    return false;
  }
  if (!dev_alloc(c, &c.d_tasks, c.tasks.size())) return false;
  if (!dev_alloc(c, &c.d_groups, c.groups.size())) return false;
  if (!dev_alloc(c, &c.d_claim, c.groups.size())) return false;
  if (!dev_alloc(c, &c.d_lags, (size_t)c.n_lags)) return false;
  if (!NFS_CUDA(c, cudaMemcpy(c.d_tasks, c.tasks.data(), sizeof(LagTask) * c.tasks.size(), cudaMemcpyHostToDevice)))
    return false;
  if (!NFS_CUDA(c, cudaMemcpy(c.d_groups, c.groups.data(), sizeof(LagGroup) * c.groups.size(), cudaMemcpyHostToDevice)))
    return false;
  if (!NFS_CUDA(c, cudaMemcpy(c.d_lags, L.data(), sizeof(int32_t) * c.n_lags, cudaMemcpyHostToDevice))) return false;
  return true;
}

void free_all(Ctx& c) {
  void* ptrs[] = {c.ring,   c.rowbuf, c.ref,       c.Fref,  c.totals, c.I2,      c.I1,      c.sums,     c.tw,     c.tw_out,
                  c.d_lags, c.perm,   c.bin_start, c.d_out, c.d_tmp,  c.d_flags, c.d_tasks, c.d_groups, c.fft_cnt, c.d_claim};
  for (void* p : ptrs)
    if (p) cudaFree(p);
  for (cudaEvent_t e : c.ev_pool) cudaEventDestroy(e);
  c.ev_pool.clear();
  if (c.own_stream && c.stream) cudaStreamDestroy(c.stream);
}

bool zero_state(Ctx& c) {
  bool ok = true;
  ok &= NFS_CUDA(c, cudaMemsetAsync(c.totals, 0, sizeof(double) * (size_t)c.n_lags * c.P, c.stream));
  ok &= NFS_CUDA(c, cudaMemsetAsync(c.I2, 0, sizeof(double) * (size_t)c.P, c.stream));
  ok &= NFS_CUDA(c, cudaMemsetAsync(c.I1, 0, sizeof(double2) * (size_t)c.P, c.stream));
  ok &= NFS_CUDA(c, cudaMemsetAsync(c.d_flags, 0, sizeof(int), c.stream));
  c.n_frames = 0;
  c.n_acc = 0;
  c.n_launches = 0;
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

// steps S5 (+ the I accumulators) for the frames transformed since the last accumulation
bool flush_pending(Ctx& c) {
  const int b = (int)(c.n_frames - c.n_acc);
  if (b <= 0) return true;
  if (c.lag_variant == 1) {  // in-library cross-check path: plain kernels
    c.n_launches += launch_accum_I(c, c.n_acc, b);
    c.n_launches += launch_lag_simple(c, c.n_acc, b);
  } else {  // k_lag_tiled also accumulates the I sums of the batch
    c.n_launches += launch_lag_tiled(c, c.n_acc, b);
  }
  if (!check_launch(c, "lag launch")) return false;
  c.n_acc = c.n_frames;
  return true;
}

}  // namespace

extern "C" {

int nfs_create_ex(nfs_ctx** out, int W, int H, const int32_t* lags, int n_lags, int n_qbins, void* cuda_stream,
                  int batch_frames) {
  if (!out) return NFS_ERR_INVALID_ARG;
  *out = nullptr;
  if (!lags || n_lags < 1 || n_qbins < 1 || n_qbins > (1 << 20) || batch_frames < 0 || batch_frames > 8192)
    return NFS_ERR_INVALID_ARG;
  if (!is_pow2(W) || !is_pow2(H) || W < 32 || H < 32 || W > 4096 || H > 4096) return NFS_ERR_INVALID_ARG;
  if (W != H) return NFS_ERR_UNSUPPORTED;
  for (int l = 0; l < n_lags; ++l)
    if (lags[l] < 1 || (l > 0 && lags[l] <= lags[l - 1])) return NFS_ERR_INVALID_ARG;
  if (n_lags > 65535 * kG) return NFS_ERR_INVALID_ARG;

  nfs_ctx* h = new (std::nothrow) nfs_ctx();
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

  int dev = 0;
  if (!NFS_CUDA(c, cudaGetDevice(&dev))) goto fail;
  cudaDeviceGetAttribute(&c.max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (cuda_stream) {
    c.stream = reinterpret_cast<cudaStream_t>(cuda_stream);
  } else {
    if (!NFS_CUDA(c, cudaStreamCreateWithFlags(&c.stream, cudaStreamNonBlocking))) goto fail;
    c.own_stream = true;
  }
  {
    // memory plan: everything is sized before the first frame arrives
    size_t free_b = 0, total_b = 0;
    if (!NFS_CUDA(c, cudaMemGetInfo(&free_b, &total_b))) goto fail;
    // default batch: 1024 frames, halved (down to 128) while the ring would take more than a third of the free memory
    while (batch_frames == 0 && c.B > 128 && (double)c.R * (double)c.P * 8.0 > (double)free_b / 3.0) {
      c.B /= 2;
      c.R = c.Lmax + c.B;
    }
    const double need = (double)c.P * ((double)c.R * 8 + 8 + (double)c.n_lags * 8 + 8 + 16 + 8) +
                        (double)fft_rowT_elems(c) * 8 +
                        (double)W * H * 4 + (double)(n_lags + 1) * n_qbins * 8 + (64 << 20);
    if (need > (double)free_b) {
      free_all(c);
      delete h;
      return NFS_ERR_OOM;
    }
  }
  if (!dev_alloc(c, &c.ring, (size_t)c.R * c.P)) goto fail;
  if (!lag_make_tensor_map(c)) {
    c.status = NFS_ERR_CUDA;
    c.cuda_err = "cuTensorMapEncodeTiled failed";
    goto fail;
  }
  if (!dev_alloc(c, &c.rowbuf, fft_rowT_elems(c))) goto fail;
  if (!dev_alloc(c, &c.ref, (size_t)W * H)) goto fail;
  if (!dev_alloc(c, &c.Fref, (size_t)c.P)) goto fail;
  if (!dev_alloc(c, &c.totals, (size_t)c.n_lags * c.P)) goto fail;
  if (!dev_alloc(c, &c.I2, (size_t)c.P)) goto fail;
  if (!dev_alloc(c, &c.I1, (size_t)c.P)) goto fail;
  if (!dev_alloc(c, &c.sums, (size_t)c.B + 1)) goto fail;
  if (!dev_alloc(c, &c.fft_cnt, 1 + 3 * (size_t)c.B)) goto fail;
  if (!dev_alloc(c, &c.d_out, (size_t)(c.n_lags + 2) * c.n_qbins)) goto fail;
  if (!dev_alloc(c, &c.d_tmp, (size_t)c.P)) goto fail;
  if (!dev_alloc(c, &c.d_flags, 1)) goto fail;
  if (!build_tables(c)) goto fail;
  if (!NFS_CUDA(c, cudaMemsetAsync(c.ring, 0, sizeof(float2) * (size_t)c.R * c.P, c.stream))) goto fail;
  if (!zero_state(c)) goto fail;
  if (!NFS_CUDA(c, cudaStreamSynchronize(c.stream))) goto fail;
  *out = h;
  return NFS_OK;

fail : {
  const int st = (c.status != NFS_OK) ? c.status : NFS_ERR_CUDA;
  const bool oom = c.cuda_err.find("out of memory") != std::string::npos;
  free_all(c);
  delete h;
  return oom ? NFS_ERR_OOM : st;
}
}

int nfs_create(nfs_ctx** out, int W, int H, const int32_t* lags, int n_lags, int n_qbins, void* cuda_stream) {
  return nfs_create_ex(out, W, H, lags, n_lags, n_qbins, cuda_stream, 0);
}

int nfs_push_frames(nfs_ctx* h, const uint16_t* d_frames, int n) {
  if (!h || !d_frames || n < 1) return NFS_ERR_INVALID_ARG;
  if ((reinterpret_cast<uintptr_t>(d_frames) & 15u) != 0) return NFS_ERR_INVALID_ARG;  // 128-bit loads
  Ctx& c = h->c;
  if (c.status != NFS_OK) return c.status;
  const int64_t fpx = (int64_t)c.W * c.H;
  int done = 0;
  while (done < n) {
    // transform as many frames as the ring has room for; accumulate whenever a full batch is pending
    const int pending = (int)(c.n_frames - c.n_acc);
    const int b = std::min(c.B - pending, n - done);
    const uint16_t* fr = d_frames + (int64_t)done * fpx;
    if (c.n_frames == 0) c.n_launches += launch_make_ref(c, fr);
    c.n_launches += launch_fft_frames(c, fr, b, c.n_frames);
    if (!check_launch(c, "fft launch")) return c.status;
    c.n_frames += b;
    done += b;
    if (c.n_frames - c.n_acc == c.B && !flush_pending(c)) return c.status;
  }
  return NFS_OK;
}

int nfs_finalize(nfs_ctx* h, double* D_q_tau, double* I_q, int64_t* counts) {
  if (!h) return NFS_ERR_INVALID_ARG;
  Ctx& c = h->c;
  if (c.status != NFS_OK) return c.status;
  if (c.n_frames < 1) return NFS_ERR_STATE;
  if (!flush_pending(c)) return c.status;
  c.n_launches += launch_bin(c);
  if (!check_launch(c, "bin launch")) return c.status;
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

int nfs_get_pair_counts(nfs_ctx* h, int64_t* n_pairs) {
  if (!h || !n_pairs) return NFS_ERR_INVALID_ARG;
  const Ctx& c = h->c;
  for (int l = 0; l < c.n_lags; ++l) n_pairs[l] = c.lags[l] < c.n_frames ? c.n_frames - c.lags[l] : 0;
  return NFS_OK;
}

static int get_plane(Ctx& c, double* out) {
  std::vector<double> tmp((size_t)c.P);
  if (!NFS_CUDA(c, cudaMemcpyAsync(tmp.data(), c.d_tmp, sizeof(double) * c.P, cudaMemcpyDeviceToHost, c.stream)))
    return c.status;
  const int st = sync_and_check(c);
  if (st != NFS_OK) return st;
  ring_to_plane(c, tmp.data(), out);
  return NFS_OK;
}

int nfs_get_D2d(nfs_ctx* h, int lag_index, double* out) {
  if (!h || !out) return NFS_ERR_INVALID_ARG;
  Ctx& c = h->c;
  if (lag_index < 0 || lag_index >= c.n_lags) return NFS_ERR_INVALID_ARG;
  if (c.status != NFS_OK) return c.status;
  if (c.n_frames < 1) return NFS_ERR_STATE;
  if (!flush_pending(c)) return c.status;
  c.n_launches += launch_D2d(c, lag_index, c.d_tmp);
  if (!check_launch(c, "D2d launch")) return c.status;
  return get_plane(c, out);
}

int nfs_get_I2d(nfs_ctx* h, double* out) {
  if (!h || !out) return NFS_ERR_INVALID_ARG;
  Ctx& c = h->c;
  if (c.status != NFS_OK) return c.status;
  if (c.n_frames < 1) return NFS_ERR_STATE;
  if (!flush_pending(c)) return c.status;
  c.n_launches += launch_I2d(c, c.d_tmp);
  if (!check_launch(c, "I2d launch")) return c.status;
  return get_plane(c, out);
}

int nfs_get_variance(nfs_ctx* h, double* V_q) {
  if (!h || !V_q) return NFS_ERR_INVALID_ARG;
  Ctx& c = h->c;
  if (c.status != NFS_OK) return c.status;
  if (c.n_frames < 1) return NFS_ERR_STATE;
  if (!flush_pending(c)) return c.status;
  c.n_launches += launch_bin(c);
  if (!check_launch(c, "bin launch")) return c.status;
  if (!NFS_CUDA(c, cudaMemcpyAsync(V_q, c.d_out + (size_t)(c.n_lags + 1) * c.n_qbins, sizeof(double) * c.n_qbins,
                                   cudaMemcpyDeviceToHost, c.stream)))
    return c.status;
  return sync_and_check(c);
}

int nfs_get_V2d(nfs_ctx* h, double* out) {
  if (!h || !out) return NFS_ERR_INVALID_ARG;
  Ctx& c = h->c;
  if (c.status != NFS_OK) return c.status;
  if (c.n_frames < 1) return NFS_ERR_STATE;
  if (!flush_pending(c)) return c.status;
  c.n_launches += launch_V2d(c, c.d_tmp);
  if (!check_launch(c, "V2d launch")) return c.status;
  return get_plane(c, out);
}

int64_t nfs_num_frames(const nfs_ctx* h) { return h ? h->c.n_frames : 0; }
int nfs_ring_capacity(const nfs_ctx* h) { return h ? h->c.R : 0; }
int64_t nfs_device_bytes(const nfs_ctx* h) { return h ? h->c.dev_bytes : 0; }
int64_t nfs_num_launches(const nfs_ctx* h) { return h ? h->c.n_launches : 0; }

int nfs_set_lag_kernel(nfs_ctx* h, int variant) {
  if (!h || variant < 0 || variant > 3) return NFS_ERR_INVALID_ARG;
  h->c.lag_variant = variant == 1 ? 1 : 0;
  h->c.lag_persistent = variant == 2 ? 0 : (variant == 3 ? 1 : -1);
  return NFS_OK;
}

int nfs_plan_lags(const int32_t* lags, int n_lags, int smem_per_sm, int smem_optin, int32_t* out, int cap) {
  if (!lags || n_lags < 1 || !out || cap < 4) return NFS_ERR_INVALID_ARG;
  for (int l = 0; l < n_lags; ++l)
    if (lags[l] < 1 || (l > 0 && lags[l] <= lags[l - 1])) return NFS_ERR_INVALID_ARG;
  Ctx c;
  c.lags.assign(lags, lags + n_lags);
  c.n_lags = n_lags;
  c.Lmax = lags[n_lags - 1];
  c.max_smem_optin = smem_optin;
  if (!lag_plan(c, smem_per_sm, kLagMinBlocks * 148, 1 << 20)) return NFS_ERR_INVALID_ARG;
  const size_t need = 4 + c.groups.size() * 23 + c.tasks.size() * 4;
  if (need > (size_t)cap) return NFS_ERR_INVALID_ARG;
  int32_t* o = out;
  *o++ = (int32_t)c.groups.size();
  *o++ = (int32_t)c.tasks.size();
  *o++ = c.lag_stages;
  *o++ = (int32_t)c.lag_smem;
  for (const LagGroup& g : c.groups) {
    *o++ = g.task0, *o++ = g.ntasks, *o++ = g.tau_min, *o++ = g.tau_max, *o++ = g.flags;
    for (int w = 0; w < 16; ++w) *o++ = g.warp_task[w];
    *o++ = g.cta0, *o++ = g.nctas;
  }
  for (const LagTask& t : c.tasks) *o++ = t.tau0, *o++ = t.cnt, *o++ = t.l0, *o++ = t.kind;
  return (int)need;
}

int nfs_set_profiling(nfs_ctx* h, int enable) {
  if (!h) return NFS_ERR_INVALID_ARG;
  h->c.prof = enable != 0;
  return NFS_OK;
}

int nfs_get_kernel_times(nfs_ctx* h, double* ms, int64_t* launches) {
  if (!h) return NFS_ERR_INVALID_ARG;
  Ctx& c = h->c;
  if (c.status != NFS_OK) return c.status;
  if (!NFS_CUDA(c, cudaStreamSynchronize(c.stream))) return c.status;
  for (size_t i = 0; i < c.ev_class.size(); ++i) {
    float t = 0.f;
    if (cudaEventElapsedTime(&t, c.ev_pool[2 * i], c.ev_pool[2 * i + 1]) == cudaSuccess) {
      c.prof_ms[c.ev_class[i]] += (double)t;
      c.prof_n[c.ev_class[i]] += 1;
    }
  }
  c.ev_class.clear();
  c.ev_used = 0;
  for (int k = 0; k < kNumKernelClasses; ++k) {
    if (ms) ms[k] = c.prof_ms[k];
    if (launches) launches[k] = c.prof_n[k];
    c.prof_ms[k] = 0.0;
    c.prof_n[k] = 0;
  }
  return NFS_OK;
}

int nfs_reset(nfs_ctx* h) {
  if (!h) return NFS_ERR_INVALID_ARG;
  Ctx& c = h->c;
  cudaStreamSynchronize(c.stream);
  cudaGetLastError();
  if (c.status == NFS_ERR_ZERO_MEAN) c.status = NFS_OK;
  if (c.status != NFS_OK) return c.status;  // a CUDA error is not recoverable by reset
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
    case NFS_ERR_UNSUPPORTED: return "unsupported configuration (W != H)";
    default: return "unknown status";
  }
}

const char* nfs_last_cuda_error(const nfs_ctx* h) { return h ? h->c.cuda_err.c_str() : ""; }

}  // extern "C"
