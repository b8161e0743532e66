/*
 * nfs_dev.h — measurement and debugging aids of the nfs-b200 library.  NOT part of the product ABI (include/nfs.h):
 * these symbols are exported only by libnfs_b200_dev.so, the build that the tests and bench.py load (same object
 * files as libnfs_b200.so plus csrc/nfs_dev.cu and the access-pattern probe csrc/nfs_probe.cu).  A context created by
 * one of the two libraries must only be passed to functions of the same library.
 */
#ifndef NFS_DEV_H_
#define NFS_DEV_H_

#include "nfs.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Flag of nfs_create_opts / nfs_create_banded: */
/*   NFS_FLAG_GUARD      debugging aid: every device buffer of the context is allocated between two 64 KB guard zones
 *                       filled with a canary byte; nfs_check_guards(ctx, &n_bad) synchronises, reads the zones back and
 *                       returns NFS_OK if they are intact, NFS_ERR_STATE otherwise (n_bad HOST: overwritten bytes; may
 *                       be NULL) — an out-of-bounds write of a kernel beside one of the library's buffers is caught
 *                       without an external tool.  NFS_ERR_STATE also if the context was created without the flag. */
#define NFS_FLAG_GUARD 2u
NFS_API int nfs_check_guards(nfs_ctx* ctx, int64_t* n_bad);

/* nfs_band_plan: host-only (no CUDA call), the same walk as the sweeps of the band schedule (nfs_create_banded in nfs.h;
 * PAPER.md:L33, Fig. 2(b)): out HOST [6] = {bands, N*, batch, OLD-window frames uploaded, NEW frames uploaded, kernel
 * launches} for a stack of n_frames frames. */
NFS_API int nfs_band_plan(int64_t n_frames, const int32_t* lags, int n_lags, int ring_frames_cap, int batch_frames,
                          int64_t* out);

/* Kernel launches enqueued by this context since create/reset (bench.py's gpu_launches). */
NFS_API int64_t nfs_num_launches(const nfs_ctx* ctx);

/* Per-kernel timing for bench.py: when enabled, every kernel launch is bracketed by a CUDA event pair
 * on the context's stream.  nfs_get_kernel_times synchronises, returns the accumulated milliseconds
 * and launch counts per class since the last call — ms/launches are HOST [NFS_NUM_KERNEL_CLASSES], in
 * the order: 0 reference set-up at the first frame (sum, reference image), 1 FFT (one persistent
 * kernel per batch: frame sums, row pass, column pass), 2 unused, 3 lag accumulation (with the I sums),
 * 4 binning — and clears them. */
#define NFS_NUM_KERNEL_CLASSES 5
NFS_API int nfs_set_profiling(nfs_ctx* ctx, int enable);
NFS_API int nfs_get_kernel_times(nfs_ctx* ctx, double* ms, int64_t* launches);

/* Measurement aid for bench.py (not part of the analysis): launches `reps` times a kernel with the memory access
 * pattern of ONE lag-accumulation launch over a batch of batch_frames frames — the 2-D TMA box copies of every pixel
 * tile's lag window into shared memory and the kernel's fp64 reductions (one per (lag, pixel) for a batch of one chunk,
 * two for longer batches; of 0.0: the accumulators keep their values) — without the arithmetic, and returns its mean duration (CUDA events on the context's stream) and the
 * algorithmic bytes P (8 (window + batch) + 16 n_lags) it moves: the ceiling of the access pattern on this device, to
 * which the real kernel's small-batch (HBM-bound) regime is compared.  Synchronises.  NFS_ERR_STATE for bin-only or
 * banded contexts. */
NFS_API int nfs_probe_lag_traffic(nfs_ctx* ctx, int batch_frames, int reps, double* ms_per_launch, double* bytes_per_launch);

/* Launch shape of the lag-accumulation kernel: 0 = chosen per batch (default), 1 = always one CTA per (pixel tile,
 * lag group), 2 = always persistent CTAs that claim pixel tiles.  The same kernel code handles the same tile either
 * way (results are bit-identical); used by the tests and by bench.py's small-batch measurement. */
NFS_API int nfs_set_launch_shape(nfs_ctx* ctx, int shape);

/* Host-only introspection of the lag plan of step S5 (which lags are accumulated
 * together); makes no CUDA call, so the host logic is testable without a GPU.  Builds the plan
 * nfs_create would build for `lags` (HOST, strictly increasing, >= 1) and frames of n_px Fourier pixels on a
 * device with n_sm SMs, `smem_per_sm` bytes of shared memory per SM and `smem_optin` bytes per CTA, and writes it
 * to out (HOST, cap int32):
 *   [n_groups, n_tasks, pipeline stages, dynamic shared memory bytes per CTA, pixels per tile (32 | 64), CTAs per SM,
 *    task slots per group (8 | 16)]
 *   per group (23 values): first task, number of tasks, tau_min, tau_max, flags (bit 0: one task of the
 *     group accumulates the I sums; bit 1: single stream, the batch's frames are the head of the window),
 *     then for task slots 0..15 the task (relative) a consumer warp of that slot runs or -1, then the
 *     first persistent CTA of the group and their number
 *   per task (4 values): smallest lag, number of lags, index of its first lag in `lags`, kind (bit 0:
 *     0 = run of consecutive lags on the register-window path, 1 = lag list; bit 1: also accumulates sum |F'|^2,
 *     bit 2: also accumulates sum F' — the two sums of the static spectrum I)
 * Returns the number of int32 written (> 0), or NFS_ERR_INVALID_ARG (bad list, cap too small, a single
 * task's lag span exceeding shared memory). */
NFS_API int nfs_plan_lags(const int32_t* lags, int n_lags, int n_px, int smem_per_sm, int smem_optin, int n_sm, int32_t* out,
                          int cap);

#ifdef __cplusplus
}
#endif
#endif /* NFS_DEV_H_ */
