// nfs_common.cuh — shared declarations of the CUDA hot path (product code; shares nothing with oracle/).
//
// Data layout in HBM.  n = W/2, P = (n+1)*H Fourier pixels per frame (half plane):
//   Fourier frame  float2[P]  = [kx = 0..n][ky = 0..H-1]  (transposed: ky fastest, FFT order), so that
//                               the column pass writes contiguous 8*H-byte rows and every row is
//                               16-byte aligned, Nyquist column included.
//   ring           float2[R][P], slot(t) = t mod R, R = Lmax + batch   (PAPER.md:L33 FIFO of image FFTs)
//   totals         double[n_lags][P]   sum over pairs of |F'_t - F'_{t+tau}|^2   ("differences area", L33)
//   ref            float[H][W]   first normalised frame r; F'_t = FFT(i_t - r)   (linearity, L31)
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>
#include <string>
#include <vector>

#include "../../include/nfs.h"
#include "../../include/nfs_dev.h"  // internal code sees the debugging aids too (NFS_FLAG_GUARD is handled at create)

namespace nfs {

// ---- lag-accumulation plan (built on the host at create, nfs_lag.cu: lag_plan) ---------------------
constexpr int kG = 13;            // lags per register-window task (window depth)
constexpr int kTaskSlots = 8;     // lag tasks per group (16 for long-window plans): one consumer warp each per 32-pixel sub-tile
constexpr int kChunk = 2 * kG;    // time steps per shared-memory pipeline stage (multiple of kG, <= 32)
constexpr int kMinStages = 2;
constexpr int kMaxStages = 8;     // pipeline depth is chosen at create from the shared memory left
constexpr int kFoldChunks = 40;   // fp32 partial sums are folded into the fp64 totals every kFoldChunks * kChunk (1040) steps
constexpr int kSparseMax = 6;     // lags per lag-list task (one LDS.64 per pair update, exact-count code paths)
constexpr int kDenseMaxWide = 5;  // lags per register-window task in a 16-slot plan (long windows): balances the runs against the lag lists
constexpr int kDenseMin = 2;      // runs of >= kDenseMin consecutive lags use the register-window path

struct LagTask {
  int tau0;  // smallest lag of the task
  int cnt;   // number of lags handled (<= kG)
  int l0;    // index of the first lag in the sorted lag list
  int kind;  // bit 0: 0 = dense run tau0..tau0+cnt-1, 1 = sparse list lags[l0..l0+cnt); bit 1: also accumulates I2
             // (sum |F'|^2); bit 2: also accumulates I1 (sum F')
};
struct LagGroup {
  int task0, ntasks;
  int tau_min, tau_max;
  int flags;  // bit 0: one task of this group accumulates the I sums (the group runs for every batch)
              // bit 1: single stream: the batch's own frames are read from the head of the window ring
  int cta0, nctas;  // persistent CTAs [cta0, cta0 + nctas) of the launch work on this group (share ~ its work)
  signed char warp_task[16];  // task (relative to task0) run by consumer warp slot w < kTaskSlots, or -1: placed so
                              // that the four SM sub-partitions (warp id mod 4) carry equal work
};

// kernel classes for the optional per-kernel CUDA-event timing (nfs_set_profiling)
enum KernelClass { kKSum = 0, kKFft = 1, kKAux = 2, kKLag = 3, kKBin = 4, kNumKernelClasses = 5 };

struct Ctx {
  int W = 0, H = 0, n = 0;  // n = W/2
  int64_t P = 0;
  int n_lags = 0, n_qbins = 0, Lmax = 0;
  int B = 0;   // internal batch (frames)
  int R = 0;   // ring slots
  int device = 0;
  int n_sm = 0;
  bool bin_only = false;  // accumulate |q|-binned totals only (no 2-D spectra kept)
  bool direct_only = false;  // NFS_FLAG_DIRECT: no neighbouring-lag recurrence, every lag accumulated as |z_s - z_o|^2
  bool guard = false;     // NFS_FLAG_GUARD: canary zones around every device buffer (nfs_check_guards)
  struct Alloc {
    void* base;         // what cudaMalloc returned
    size_t user_bytes;  // the buffer's size rounded up to 256 bytes
  };
  std::vector<Alloc> allocs;
  // Out-of-core band schedule (Fig. 2(b) L37): the device holds only `ring cap` Fourier frames, fewer
  // than Lmax + batch.  The lags are cut into bands of band_width = N* lags (the paper's FIFO length); band 0 is
  // accumulated while the frames stream through the ring (the "first triangle" and its diagonal), every Fourier frame
  // is also kept in pinned host memory, and the further bands are swept at finalize: per band a window of N* + batch
  // OLD frames (the FIFO, in `ring`) and a batch of NEW frames (the "current image area", in `ringN`) are uploaded
  // again from the host store.
  int band_width = 0;           // N*; 0: everything fits (Fig. 2(a)), no host store
  int n_bands = 1;
  int RN = 0;                   // slots of ringN (= batch)
  float2* ringN = nullptr;      // ring + R * P
  CUtensorMap ringN_map;
  float2* h_store = nullptr;    // pinned host memory [max_frames][P]
  int64_t max_frames = 0;
  std::vector<int> band_g0;     // [n_bands + 1] first lag group of each band
  std::vector<int> band_l0;     // [n_bands + 1] index of the first lag of each band
  int64_t swept_frames = -1;    // the sweeps of bands >= 1 are up to date for this many frames
  bool ring_dirty = false;      // the sweeps overwrote the streaming ring: restored from the host store at the next push
  int64_t h2d_frames = 0, d2h_frames = 0;  // Fourier frames moved by the band schedule (the paper's N_FFT counts the uploads)
  std::vector<int32_t> lags;
  std::vector<int64_t> counts;  // full-plane pixel count per bin
  cudaStream_t stream = nullptr;
  bool own_stream = false;
  // time-chunk sharding over several contexts / GPUs: halo frames precede this context's own frames
  // (they are transformed and paired with the own frames, but are no later frame of a pair and not in the I sums);
  // after nfs_import_partials the sums are those of all contexts (`merged`): pair and frame counts come with them
  int64_t n_halo = 0;
  bool merged = false;
  std::vector<int64_t> merged_pairs;  // [n_lags]
  int64_t merged_frames = 0;
  long long* d_npairs = nullptr;      // [n_lags] divisors of the binning kernel
  int64_t n_frames = 0;  // frames pushed (all transformed into the ring), halo included
  int64_t n_acc = 0;     // of those, frames whose pairs are already in the totals
  int64_t n_launches = 0;
  int status = 0;  // sticky
  std::string cuda_err;
  int64_t dev_bytes = 0;
  int max_smem_optin = 0;

  // device memory
  float2* ring = nullptr;
  CUtensorMap ring_map;          // 2-D TMA descriptor of the ring (nfs_lag.cu): box = tile pixels x kChunk slots
  float2* rowbuf = nullptr;      // [slots][P] output of the row pass (transposed, L2 resident)
  float* ref = nullptr;          // [H][W]
  float2* Fref = nullptr;        // [P] unitary FFT of ref
  double* totals = nullptr;      // [n_lags][P]; bin-only mode: scratch [max lags of a group][P]
  double* totals_b = nullptr;    // bin-only mode: [n_lags][n_qbins] weighted sums over the bin's pixels
  double* I2 = nullptr;          // [P]  sum_t |F'_t|^2
  double2* I1 = nullptr;         // [P]  sum_t F'_t
  unsigned long long* sums = nullptr;  // [B + 1] exact pixel sums of the frames of a batch; [B] = S_0
  unsigned int* fft_cnt = nullptr;     // work-queue head and per-frame completion counters of k_fft
  int fft_grid = 0;                    // CTAs of the persistent FFT kernel (set at create)
  float2* tw = nullptr;          // inner twiddle table (nfs_fft.cu)
  float2* tw_out = nullptr;      // outer twiddle table, W > 1024 only
  int32_t* d_lags = nullptr;     // [n_lags]
  uint32_t* perm = nullptr;      // [n_binned] pixel index | (weight-2 flag << 31), grouped by bin
  int32_t* bin_start = nullptr;  // [n_qbins + 1]
  double* d_out = nullptr;       // [(n_lags + 2)][n_qbins] binned results: D rows, I row, V row
  double* d_fit = nullptr;       // [4][n_qbins] Eq. 1 fit: A, C, Gamma, chi2
  double* d_tmp = nullptr;       // [P] scratch for the 2-D getters
  int* d_flags = nullptr;        // [1] bit0 = zero-mean frame seen
  LagTask* d_tasks = nullptr;
  LagGroup* d_groups = nullptr;
  int* d_claim = nullptr;        // [n_groups] next pixel tile of each group, zeroed before every persistent launch
  int lag_stages = kMinStages;   // pipeline stages of k_lag_tiled (chosen by lag_plan)
  int lag_tpx = 32;              // Fourier pixels per CTA tile: 32 or 64
  int lag_slots = kTaskSlots;    // task slots per group: 8, or 16 (one 32-pixel CTA of 16 consumer warps per SM)
  int lag_ctas_per_sm = 1;       // resident CTAs per SM the plan counts on
  int lag_grid = 0;              // persistent CTAs of k_lag_tiled (sum of the groups' shares)
  int lag_shape = 0;             // 0: chosen per launch (launch_lag_tiled); 1 / 2: forced one-tile / persistent
  size_t lag_smem = 0;           // dynamic shared memory of k_lag_tiled
  int max_group_lags = 0;        // most lags in one group (bin-only scratch rows)
  std::vector<LagTask> tasks;
  std::vector<LagGroup> groups;

  // per-kernel timing: pairs of events recorded on the context's stream around each launch
  bool prof = false;
  std::vector<cudaEvent_t> ev_pool;
  size_t ev_used = 0;
  std::vector<int> ev_class;  // class of pair i (events 2i, 2i+1)
  double prof_ms[kNumKernelClasses] = {0, 0, 0, 0, 0};
  int64_t prof_n[kNumKernelClasses] = {0, 0, 0, 0, 0};
};

// frames in the I sums, and frame pairs accumulated at lag index l (N - tau for a whole stack)
inline int64_t frames_in_I(const Ctx& c) { return c.merged ? c.merged_frames : c.n_frames - c.n_halo; }
inline int64_t pair_count(const Ctx& c, int l) {
  if (c.merged) return c.merged_pairs[(size_t)l];
  const int64_t own = c.n_frames - c.n_halo;  // later frames s = n_halo .. n_frames-1; pair (s - tau, s) exists iff s >= tau
  const int64_t missing = std::max<int64_t>(0, (int64_t)c.lags[(size_t)l] - c.n_halo);
  return std::max<int64_t>(0, own - missing);
}

// record the first CUDA error of the context (sticky)
inline bool cuda_ok(Ctx& c, cudaError_t e, const char* what) {
  if (e == cudaSuccess) return true;
  if (c.status == NFS_OK) {
    c.status = NFS_ERR_CUDA;
    c.cuda_err = std::string(what) + ": " + cudaGetErrorString(e);
  }
  return false;
}
#define NFS_CUDA(c, call) ::nfs::cuda_ok((c), (call), #call)

// RAII: records an event pair around the launches enqueued in its scope when profiling is on
struct ProfScope {
  Ctx& c;
  cudaEvent_t stop = nullptr;
  ProfScope(Ctx& ctx, int cls) : c(ctx) {
    if (!c.prof) return;
    while (c.ev_pool.size() < c.ev_used + 2) {
      cudaEvent_t e;
      if (!NFS_CUDA(c, cudaEventCreate(&e))) return;
      c.ev_pool.push_back(e);
    }
    cudaEvent_t start = c.ev_pool[c.ev_used];
    stop = c.ev_pool[c.ev_used + 1];
    c.ev_used += 2;
    c.ev_class.push_back(cls);
    NFS_CUDA(c, cudaEventRecord(start, c.stream));
  }
  ~ProfScope() {
    if (stop) NFS_CUDA(c, cudaEventRecord(stop, c.stream));
  }
};

// ---- kernel launchers (each returns the number of kernel launches it enqueued; CUDA errors go to c.status) ----
// nfs_fft.cu
bool fft_configure(Ctx& c);                                       // once at create: kernel attributes, grid size
int launch_make_ref(Ctx& c, const uint16_t* frame0);              // S_0, ref = i_0, Fref = FFT(ref)
int launch_fft_frames(Ctx& c, const uint16_t* frames, int nf, int64_t t_first);  // ring[t_first..] = FFT(i_t - ref)
size_t fft_rowT_elems(const Ctx& c);                              // float2 elements of the row-pass buffer
size_t fft_cnt_elems(const Ctx& c);                               // unsigned ints of the work-queue counters
// nfs_lag.cu
int launch_lag_tiled(Ctx& c, int64_t t0, int b, int band = 0);  // band > 0: a sweep of the band schedule (NEW frames from ringN)
// host only (no CUDA call): tasks, groups, tile width, pipeline depth from the lag list, the shared memory per SM and
// c.max_smem_optin; false if a lag group cannot fit shared memory
bool lag_plan(Ctx& c, int smem_per_sm, int n_sm, int64_t P);
bool lag_configure(Ctx& c);        // once at create, after the ring is allocated: tensor map, kernel attributes
// nfs_probe.cu (measurement aid): the traffic of one small-batch lag launch without its arithmetic
int launch_lag_probe(Ctx& c, int b, double* bytes);
// nfs_bin.cu
int launch_bin(Ctx& c);                      // d_out = azimuthal means of D (rows 0..n_lags-1), I (row n_lags), V (row n_lags+1)
int launch_fit_eq1(Ctx& c);                  // after launch_bin: d_fit = per-|q| fit of Eq. 1 to the binned D
int launch_bin_accumulate(Ctx& c, int l_first, int n_rows);  // bin-only mode: totals_b[l_first..] += binned scratch rows
int launch_absolute_I(Ctx& c, double* d_S2, double2* d_S1);  // S2 = sum |F_t|^2, S1 = sum F_t over the context's own frames
int launch_I2d(Ctx& c, double* d_dst);       // d_dst[P] = I2d in ring layout
int launch_V2d(Ctx& c, double* d_dst);       // d_dst[P] = V2d (variance form) in ring layout
int launch_D2d(Ctx& c, int l, double* d_dst);

// ---- shared by nfs_api.cu (product ABI) and nfs_dev.cu (measurement / debugging ABI, dev build only) ----------------
}  // namespace nfs

struct nfs_ctx {
  nfs::Ctx c;
};

namespace nfs {

// guard zones of NFS_FLAG_GUARD (nfs_dev.h): bytes on either side of every device buffer, and their canary value
constexpr size_t kGuardBytes = 64 << 10;
constexpr int kGuardByte = 0xA5;

// every entry point that touches the device runs on the context's device
inline bool enter(Ctx& c) {
  if (c.status != NFS_OK) return false;
  int dev = -1;
  if (!NFS_CUDA(c, cudaGetDevice(&dev))) return false;
  if (dev != c.device && !NFS_CUDA(c, cudaSetDevice(c.device))) return false;
  return true;
}

inline bool lags_ok(const int32_t* lags, int n_lags) {
  if (!lags || n_lags < 1) return false;
  for (int l = 0; l < n_lags; ++l)
    if (lags[l] < 1 || (l > 0 && lags[l] <= lags[l - 1])) return false;
  return true;
}


// ---- out-of-core band schedule (Fig. 2(b) L37) ----------------------------------------------------
// Memory plan for a device that holds only `cap` Fourier frames: batch b, band width N* = cap - 2 b (a window of
// N* + b OLD frames and b NEW frames).  Returns false if no band fits.
inline bool band_memory_plan(int cap, int batch_frames, int* b_out, int* nstar_out) {
  int b = batch_frames > 0 ? batch_frames : std::min(1024, cap / 4);
  b = std::max(1, std::min(b, 8192));
  const int nstar = cap - 2 * b;
  if (nstar < 1) return false;
  *b_out = b;
  *nstar_out = nstar;
  return true;
}

// The sweeps of bands 1 .. n_bands-1 over a stack of N frames, as a sequence of uploads and launches.  Band k holds
// the requested lags in (k N*, (k+1) N*], smallest tmin, largest tmax.  Its sweep walks the frames s = tmin .. N-1 in
// batches of b: the batch goes into the NEW ring, the OLD frames s - tmax .. s - tmin it pairs with are kept in the
// OLD ring, every frame of the window being uploaded once per band (the paper's FIFO: "one diagonal is filled by
// subsequently replacing one FIFO image and uploading one 'current image'").  The same walk serves the device (uploads
// and kernel launches) and the host-only transfer count of nfs_band_plan.
template <typename UploadOld, typename UploadNew, typename Launch>
bool band_sweeps(int64_t N, int b, int n_bands, const std::vector<int>& band_l0, const std::vector<int32_t>& lags,
                 UploadOld&& upload_old, UploadNew&& upload_new, Launch&& launch) {
  for (int k = 1; k < n_bands; ++k) {
    const int l0 = band_l0[(size_t)k], l1 = band_l0[(size_t)k + 1];
    if (l1 <= l0) continue;  // no requested lag in this band
    const int64_t tmin = lags[(size_t)l0], tmax = lags[(size_t)l1 - 1];
    int64_t old_next = -1;  // first OLD frame not yet in the OLD ring
    for (int64_t t0 = tmin; t0 < N; t0 += b) {
      const int bb = (int)std::min<int64_t>(b, N - t0);
      const int64_t lo = std::max<int64_t>(0, t0 - tmax), hi = t0 + bb - 1 - tmin;  // OLD frames lo .. hi
      const int64_t from = std::max(lo, old_next);
      if (hi >= from && !upload_old(from, hi + 1)) return false;
      old_next = std::max(old_next, hi + 1);
      if (!upload_new(t0, t0 + bb)) return false;
      if (!launch(t0, bb, k)) return false;
    }
  }
  return true;
}

// Nothing may throw across the C boundary: allocation failures of the host-side containers become NFS_ERR_OOM.
#define NFS_GUARDED(expr)            \
  try {                              \
    return (expr);                   \
  } catch (const std::bad_alloc&) {  \
    return NFS_ERR_OOM;              \
  } catch (...) {                    \
    return NFS_ERR_STATE;            \
  }


}  // namespace nfs
