// nfs_dev.cu — the entry points of include/nfs_dev.h: measurement and debugging aids (per-kernel timing, launch counts,
// guard zones, lag-plan and band-plan introspection, launch-shape override, the access-pattern probe).  Linked only into
// libnfs_b200_dev.so, which the tests and bench.py load; the product library libnfs_b200.so does not contain this file
// (nor nfs_probe.cu) and exports none of these symbols.
#include <math.h>

#include "nfs_common.cuh"

using namespace nfs;

static int band_plan_impl(int64_t n_frames, const int32_t* lags, int n_lags, int ring_frames_cap, int batch_frames, int64_t* out) {
  if (!lags_ok(lags, n_lags) || !out || n_frames < 1 || ring_frames_cap < 1) return NFS_ERR_INVALID_ARG;
  int b = 0, nstar = 0;
  if (!band_memory_plan(ring_frames_cap, batch_frames, &b, &nstar) || lags[0] > nstar) return NFS_ERR_INVALID_ARG;
  const int n_bands = (lags[n_lags - 1] - 1) / nstar + 1;
  std::vector<int32_t> L(lags, lags + n_lags);
  std::vector<int> l0((size_t)n_bands + 1, n_lags);
  for (int l = n_lags - 1; l >= 0; --l)
    for (int k = 0; k <= (L[(size_t)l] - 1) / nstar; ++k) l0[(size_t)k] = l;
  int64_t up_old = 0, up_new = 0, launches = 0;
  band_sweeps(
      n_frames, b, n_bands, l0, L, [&](int64_t f0, int64_t f1) { up_old += f1 - f0; return true; },
      [&](int64_t f0, int64_t f1) { up_new += f1 - f0; return true; }, [&](int64_t, int, int) { ++launches; return true; });
  out[0] = n_bands, out[1] = nstar, out[2] = b, out[3] = up_old, out[4] = up_new, out[5] = launches;
  return NFS_OK;
}
int nfs_band_plan(int64_t n_frames, const int32_t* lags, int n_lags, int ring_frames_cap, int batch_frames, int64_t* out) {
  NFS_GUARDED(band_plan_impl(n_frames, lags, n_lags, ring_frames_cap, batch_frames, out))
}


static int probe_impl(nfs_ctx* h, int batch_frames, int reps, double* ms_per_launch, double* bytes_per_launch) {
  if (!h || batch_frames < 1 || reps < 1 || !ms_per_launch) return NFS_ERR_INVALID_ARG;
  Ctx& c = h->c;
  if (!enter(c)) return c.status;
  if (c.bin_only || c.band_width > 0) return NFS_ERR_STATE;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (!NFS_CUDA(c, cudaEventCreate(&e0))) return c.status;
  if (!NFS_CUDA(c, cudaEventCreate(&e1))) {
    cudaEventDestroy(e0);
    return c.status;
  }
  double bytes = 0.0;
  launch_lag_probe(c, batch_frames, &bytes);  // warm-up
  NFS_CUDA(c, cudaEventRecord(e0, c.stream));
  for (int r = 0; r < reps; ++r) c.n_launches += launch_lag_probe(c, batch_frames, &bytes);
  NFS_CUDA(c, cudaEventRecord(e1, c.stream));
  NFS_CUDA(c, cudaStreamSynchronize(c.stream));
  float ms = 0.f;
  NFS_CUDA(c, cudaEventElapsedTime(&ms, e0, e1));
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  *ms_per_launch = (double)ms / reps;
  if (bytes_per_launch) *bytes_per_launch = bytes;
  return c.status;
}
int nfs_probe_lag_traffic(nfs_ctx* h, int batch_frames, int reps, double* ms_per_launch, double* bytes_per_launch) {
  NFS_GUARDED(probe_impl(h, batch_frames, reps, ms_per_launch, bytes_per_launch))
}

static int guards_impl(nfs_ctx* h, int64_t* n_bad) {
  if (!h) return NFS_ERR_INVALID_ARG;
  Ctx& c = h->c;
  if (!c.guard) return NFS_ERR_STATE;
  if (!enter(c)) return c.status;
  if (!NFS_CUDA(c, cudaStreamSynchronize(c.stream))) return c.status;
  std::vector<unsigned char> buf(kGuardBytes);
  int64_t bad = 0;
  for (const Ctx::Alloc& a : c.allocs) {
    const char* base = static_cast<const char*>(a.base);
    for (int side = 0; side < 2; ++side) {  // the zone in front of the buffer, then the one behind its 256-byte rounded end
      if (!NFS_CUDA(c, cudaMemcpy(buf.data(), base + (side ? kGuardBytes + a.user_bytes : 0), kGuardBytes, cudaMemcpyDeviceToHost)))
        return c.status;
      for (unsigned char v : buf) bad += v != (unsigned char)kGuardByte;
    }
  }
  if (n_bad) *n_bad = bad;
  return bad == 0 ? NFS_OK : NFS_ERR_STATE;
}
int nfs_check_guards(nfs_ctx* h, int64_t* n_bad) { NFS_GUARDED(guards_impl(h, n_bad)) }


int nfs_set_launch_shape(nfs_ctx* h, int shape) {
  if (!h || shape < 0 || shape > 2) return NFS_ERR_INVALID_ARG;
  h->c.lag_shape = shape;
  return NFS_OK;
}

static int plan_impl(const int32_t* lags, int n_lags, int n_px, int smem_per_sm, int smem_optin, int n_sm, int32_t* out,
                     int cap) {
  if (!lags_ok(lags, n_lags) || !out || cap < 7 || n_px < 32 || n_sm < 1) return NFS_ERR_INVALID_ARG;
  Ctx c;
  c.lags.assign(lags, lags + n_lags);
  c.n_lags = n_lags;
  c.Lmax = lags[n_lags - 1];
  c.max_smem_optin = smem_optin;
  if (!lag_plan(c, smem_per_sm, n_sm, (int64_t)n_px)) return NFS_ERR_INVALID_ARG;
  const size_t need = 7 + c.groups.size() * 23 + c.tasks.size() * 4;
  if (need > (size_t)cap) return NFS_ERR_INVALID_ARG;
  int32_t* o = out;
  *o++ = (int32_t)c.groups.size();
  *o++ = (int32_t)c.tasks.size();
  *o++ = c.lag_stages;
  *o++ = (int32_t)c.lag_smem;
  *o++ = c.lag_tpx;
  *o++ = c.lag_ctas_per_sm;
  *o++ = c.lag_slots;
  for (const LagGroup& g : c.groups) {
    *o++ = g.task0, *o++ = g.ntasks, *o++ = g.tau_min, *o++ = g.tau_max, *o++ = g.flags;
    for (int w = 0; w < 16; ++w) *o++ = g.warp_task[w];
    *o++ = g.cta0, *o++ = g.nctas;
  }
  for (const LagTask& t : c.tasks) *o++ = t.tau0, *o++ = t.cnt, *o++ = t.l0, *o++ = t.kind;
  return (int)need;
}
int nfs_plan_lags(const int32_t* lags, int n_lags, int n_px, int smem_per_sm, int smem_optin, int n_sm, int32_t* out, int cap) {
  NFS_GUARDED(plan_impl(lags, n_lags, n_px, smem_per_sm, smem_optin, n_sm, out, cap))
}

int nfs_set_profiling(nfs_ctx* h, int enable) {
  if (!h) return NFS_ERR_INVALID_ARG;
  h->c.prof = enable != 0;
  return NFS_OK;
}

static int times_impl(nfs_ctx* h, double* ms, int64_t* launches) {
  if (!h) return NFS_ERR_INVALID_ARG;
  Ctx& c = h->c;
  if (!enter(c)) return c.status;
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
int nfs_get_kernel_times(nfs_ctx* h, double* ms, int64_t* launches) { NFS_GUARDED(times_impl(h, ms, launches)) }


int64_t nfs_num_launches(const nfs_ctx* h) { return h ? h->c.n_launches : 0; }
