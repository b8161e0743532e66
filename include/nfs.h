/*
 * nfs.h — C ABI of the B200 (sm_100a) hot path of the double-frame differential analysis of
 * dynamic near-field-scattering / shadowgraph / DDM image stacks (arxiv 1209.3362,
 * Cerchiari, Croccolo, Cardinaux, Scheffold).  Citations are lines of /root/reference/PAPER.md.
 *
 * What the library computes (the paper's method; readings R1-R18 in DESIGN.md §3):
 *   1. every pushed uint16 frame is normalised by its spatial mean
 *   2. and Fourier-transformed exactly once, 2-D real-to-complex, unitary      (L25, L31)
 *   3. the transformed frames live in a ring buffer in HBM — the role of the
 *      paper's G-RAM FIFO of image FFTs, Fig. 2(a)                             (L33, L37)
 *   4. for every requested lag tau the structure function
 *        D2d(k,tau) = < |F_t(k) - F_{t+tau}(k)|^2 >_t   over all N-tau pairs   (L21, L25, L31-33)
 *      is accumulated in Fourier space (linearity, L31), and the static spectrum
 *        I2d(k) = < |F_t(k)|^2 >_t                                             (R9)
 *   5. both are azimuthally averaged into n_qbins uniform |q| bins on [0, q_Nyquist),
 *      DC pixel excluded, bin index by exact integer arithmetic                (L25; R6, R7)
 *
 * Accuracy.  Transforms and pair differences are fp32, partial sums are folded into fp64.  Binned D and
 * I agree with the fp64 definition to 1e-4 relative, D2d per pixel to 1e-3 wherever D2d > 1e-6 of its maximum.  A lag
 * that opens a run of consecutive requested lags (or stands alone) is summed directly and carries only its own relative
 * rounding; the further lags of a run are built from their neighbour, and their ABSOLUTE error at pixel k is bounded by
 *     1e-6 * Z(k) * E(k),   Z = max_t |F_t(k) - F_0(k)|,   E = max_t |F_t(k) - F_{t-1}(k)|,
 * i.e. it scales with how far the stack has wandered from its first frame, not with D2d(k,tau) itself.  For stationary
 * fluctuations (Z^2 of the order of the plateau) this is far inside the relative bars above; for a stack that drifts
 * away from frame 0 by more than ~1000 frame-to-frame increments at a pixel, small-lag values there lose relative
 * accuracy accordingly (create the context with NFS_FLAG_DIRECT if that matters).
 *
 * Every step runs in hand-written CUDA kernels; there is no CPU fallback and no cuFFT.
 * One context = one CUDA device (the one current at nfs_create; later calls switch to it) = one CUDA
 * stream = not thread-safe; contexts are independent; no global state.  (Measurement and debugging aids — per-kernel
 * timing, launch counts, guard zones, plan introspection, the traffic probe — are NOT part of this ABI: they are declared
 * in include/nfs_dev.h and exported only by the test/bench build libnfs_b200_dev.so.)
 * All functions return 0 (NFS_OK) or a negative nfs_status; nothing throws or aborts across
 * this boundary (a failed host allocation inside the library returns NFS_ERR_OOM).  Errors NFS_ERR_CUDA
 * and NFS_ERR_ZERO_MEAN are sticky: once raised every later call on the context returns them until
 * nfs_reset() (which clears NFS_ERR_ZERO_MEAN only; a CUDA error is final).
 */
#ifndef NFS_H_
#define NFS_H_

#include <stdint.h>

#if defined(__GNUC__)
#define NFS_API __attribute__((visibility("default")))
#else
#define NFS_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nfs_ctx nfs_ctx; /* opaque, owned by the library */

typedef enum nfs_status {
  NFS_OK = 0,
  NFS_ERR_INVALID_ARG = -1, /* NULL pointer; W or H not a power of two in [32,4096]; n_lags < 1 or > 65533; lags
                               not strictly increasing or < 1; n_qbins < 1; n < 1; d_frames not 16-byte aligned;
                               index out of range                                                   */
  NFS_ERR_OOM = -2,         /* ring + accumulators do not fit the free device memory (checked at create) */
  NFS_ERR_CUDA = -3,        /* first failing CUDA call (sticky)                                        */
  NFS_ERR_ZERO_MEAN = -4,   /* a pushed frame summed to zero: its normalisation (L21) is undefined.
                               Detected on the device, surfaced by the next synchronising call (sticky) */
  NFS_ERR_STATE = -5,       /* call not valid in this state (finalize or a getter before any own frame — halo
                               frames do not count; a 2-D difference spectrum asked of a bin-only context) */
  NFS_ERR_UNSUPPORTED = -6, /* W != H (all of the paper's sizes, L33, are square); the band schedule asked
                               for together with NFS_FLAG_BIN_ONLY                                     */
  NFS_ERR_TOO_LARGE = -7    /* nfs_azimuthal_mean_static only: n_qbins exceeds NFS_STATIC_MAX_QBINS, the size its
                               fixed scratch array was built for                                       */
} nfs_status;

/*
 * nfs_create — plan memory and build the tables ("optimize memory allocation prior to
 * starting the calculations"; here the trivial alpha=1 case of Fig. 2(a): ring = Lmax + batch frames).
 *   out       HOST  receives the context.
 *   W,H             frame size in pixels, powers of two in [32,4096], W == H.
 *   lags      HOST  [n_lags] lags in frames, >= 1, strictly increasing (copied).
 *   n_qbins         number of |q| bins on [0, pi rad/px).
 *   cuda_stream     a cudaStream_t cast to void*, or NULL for a library-owned stream.  All device
 *                   work of this context is enqueued on it.
 * nfs_create_ex additionally fixes the internal batch size, 1..8192 (0 = default: 1024, halved down to
 * 128 while the ring would take more than a third of the free device memory): pushed frames are
 * transformed into the ring at once, their frame pairs are accumulated whenever `batch` frames are
 * pending (and at every finalize/getter).  Ring capacity is Lmax + batch frames of H*(W/2+1) complex64.
 * Whatever the batch, fp32 partial sums never span more than 1040 frames before they are folded into
 * the fp64 totals.
 * nfs_create_opts additionally takes flags:
 *   NFS_FLAG_BIN_ONLY   keep only the |q|-binned sums of the difference spectra ("store the
 *                       entire 2D power spectra, which might be unnecessary"): the [n_lags][H][W/2+1] fp64
 *                       accumulators (4.2 GB for 1000 lags at 1024^2) shrink to a scratch for one group of
 *                       <= 104 lags plus [n_lags][n_qbins]; nfs_finalize returns the same D, I, counts (same
 *                       fixed summation order within a bin: run-to-run bit-identical); nfs_get_D2d returns
 *                       NFS_ERR_STATE.
 *   NFS_FLAG_DIRECT     accumulate every lag by the plain difference form sum |F_t - F_{t+tau}|^2 and never through
 *                       the neighbouring-lag recurrence: each lag then carries only its own relative rounding (exact
 *                       zeros stay exact; no error term that grows with the stack's excursion from its first frame,
 *                       see "Accuracy" above), at about three times the lag-accumulation time for runs of consecutive
 *                       lags (measured on a B200: 40.6 instead of 18.4 ms per 1024^2 x 2000-frame, 100-lag stack).  For stacks
 *                       that drift far from frame 0, or when D(q,tau) is wanted far below its plateau.
 */
#define NFS_FLAG_BIN_ONLY 1u
#define NFS_FLAG_DIRECT 4u /* (2u is NFS_FLAG_GUARD of nfs_dev.h) */
NFS_API int nfs_create(nfs_ctx** out, int W, int H, const int32_t* lags, int n_lags, int n_qbins, void* cuda_stream);
NFS_API int nfs_create_ex(nfs_ctx** out, int W, int H, const int32_t* lags, int n_lags, int n_qbins, void* cuda_stream,
                          int batch_frames);
NFS_API int nfs_create_opts(nfs_ctx** out, int W, int H, const int32_t* lags, int n_lags, int n_qbins, void* cuda_stream,
                            int batch_frames, unsigned flags);

/*
 * nfs_create_banded — the out-of-core schedule of PAPER.md:L33 and Fig. 2(b) (L37) for lag windows that exceed the
 * device memory one is willing to spend: "if the number of images to be analyzed exceeds the G-RAM capacity then data
 * has to be transferred multiple times ... data transfer can be optimized by organizing the memory as a First-In-
 * First-Out (FIFO) queue ... N - 1 = alpha N* + beta".
 *   ring_frames_cap   Fourier frames the device may hold (0 = no limit: identical to nfs_create_opts).  If it is
 *                     smaller than Lmax + batch, the lags are cut into bands of N* = cap - 2 batch lags (batch =
 *                     batch_frames, or min(1024, cap / 4) if 0).  Band 0 (lags <= N*) is accumulated while the frames
 *                     stream through the ring, as in Fig. 2(a) ("the first triangle"); every Fourier frame is also
 *                     copied once to pinned HOST memory owned by the library; the further bands ("diagonals") are
 *                     swept at nfs_finalize / the getters: per band a FIFO window of N* + batch OLD frames and a
 *                     "current image area" of `batch` NEW frames are uploaded again from that store, every frame at
 *                     most twice per band (the paper's 2 alpha N transfers; its N_FFT = N (2 alpha - 3 + 2 / alpha)
 *                     counts N - N* steps of two uploads for every further band, this schedule stops a band where its
 *                     pairs end).  Frames are transformed once: what is uploaded again are Fourier frames.
 *   max_frames        frames the host store is sized for (> 0 in band mode; pushing more returns NFS_ERR_INVALID_ARG).
 * Requirements in band mode: the smallest requested lag <= N*; no NFS_FLAG_BIN_ONLY (NFS_ERR_UNSUPPORTED).  Results
 * are those of nfs_create up to fp32 partial-sum rounding (other batch boundaries).  nfs_finalize stays a
 * non-destructive snapshot: the bands are rebuilt from the store at each finalize that sees new frames, and the
 * streaming ring is restored from the store at the next push.
 * nfs_get_transfer_counts: out HOST [4] = {bands alpha, band width N* (0: not banded), Fourier frames uploaded
 * host -> device so far, Fourier frames downloaded device -> host so far}.
 */
NFS_API int nfs_create_banded(nfs_ctx** out, int W, int H, const int32_t* lags, int n_lags, int n_qbins, void* cuda_stream,
                              int batch_frames, unsigned flags, int ring_frames_cap, int64_t max_frames);
NFS_API int nfs_get_transfer_counts(const nfs_ctx* ctx, int64_t* out);

/*
 * nfs_push_frames — steps 1-4 for n more frames.
 *   d_frames  DEVICE [n][H][W] uint16, row-major, x fastest, pitch W, no padding, 16-byte aligned (the
 *             kernels read it with 128-bit loads; anything else returns NFS_ERR_INVALID_ARG).
 * Stream-ordered and asynchronous to the host: d_frames must stay valid and unmodified until the
 * work enqueued by this call on the context's stream has run (record an event after the call).
 * Frames are numbered in push order; results do not depend on how a stack is split across calls
 * (batches are cut by frame number, not by call; an interleaved finalize/getter cuts a batch early,
 * which changes fp32 partial-sum rounding only, <= 1e-6 relative).
 */
NFS_API int nfs_push_frames(nfs_ctx* ctx, const uint16_t* d_frames, int n);

/*
 * Time-chunk sharding over several contexts, one per GPU (the path of PAPER.md:L31-33 is a sum over
 * frame pairs, so it splits by the later frame of each pair).  Context g takes the frames [g N / G, (g+1) N / G) of the
 * stack as its own and, first, the Lmax frames before them as a halo:
 *   nfs_push_halo      d_frames DEVICE [n][H][W] as in nfs_push_frames.  Halo frames are normalised, transformed and
 *                      kept in the ring, and are paired with the own frames that follow as the EARLIER frame of a
 *                      pair; they are never the later frame of a pair, do not enter I(q) and are not counted.  Only
 *                      before the first own frame, at most Lmax frames in total (NFS_ERR_STATE otherwise; not in
 *                      band mode).  nfs_get_pair_counts then reports the pairs this context holds.
 *   nfs_partials_count doubles in a partial-sum buffer of this context.
 *   nfs_export_partials d_buf DEVICE [nfs_partials_count]: the context's sums in a form that adds up over contexts:
 *                      pair sums per lag and pixel (per lag and |q| bin for NFS_FLAG_BIN_ONLY), sum |F_t|^2 and
 *                      sum F_t over the own frames (absolute: independent of the context's reference frame), pair
 *                      counts per lag, own-frame count.  Synchronises the stream.  A context without own frames (the
 *                      rank of an empty time chunk, or one that has only seen its halo) exports zeros, so that it can
 *                      take part in the all-reduce like every other rank; it may import the total as well.
 *   nfs_import_partials d_buf DEVICE: replaces the context's sums by the buffer's — the caller has added the buffers
 *                      of all contexts (one all-reduce(sum), e.g. ncclAllReduce over NVLink).
 *                      Afterwards nfs_finalize and the getters return the result of the whole stack (counts and
 *                      divisors come from the buffer); pushing more frames, exporting, and a second import return
 *                      NFS_ERR_STATE until nfs_reset.
 * Export and import return NFS_ERR_STATE on a context created with a band schedule (nfs_create_banded with a binding
 * ring_frames_cap): the two ways of handling a stack that does not fit one device's memory are not combined.
 */
NFS_API int nfs_push_halo(nfs_ctx* ctx, const uint16_t* d_frames, int n);
NFS_API int64_t nfs_partials_count(const nfs_ctx* ctx);
NFS_API int nfs_export_partials(nfs_ctx* ctx, double* d_buf);
NFS_API int nfs_import_partials(nfs_ctx* ctx, const double* d_buf);

/*
 * nfs_finalize — step 5 ("azimuthally averaged power spectra") for the N frames pushed
 * so far.  Synchronises the stream; non-destructive snapshot: pushing may continue afterwards.
 *   D_q_tau   HOST [n_lags][n_qbins] double   mean of D2d over bin b; rows with tau >= N are 0.
 *   I_q       HOST [n_qbins] double           mean of I2d over bin b.
 *   counts    HOST [n_qbins] int64            full-plane pixel count of each bin (data independent).
 * Empty bins hold 0.0 / 0.  Any of the three may be NULL to skip it.
 */
NFS_API int nfs_finalize(nfs_ctx* ctx, double* D_q_tau, double* I_q, int64_t* counts);

/* n_pairs HOST [n_lags]: N - tau, or 0 when tau >= N (N(N-1)/2 pairs over N-1 lags).  Host-only;
 * returns the sticky error of the context if one is set. */
NFS_API int nfs_get_pair_counts(nfs_ctx* ctx, int64_t* n_pairs);

/* Averaged 2-D spectra on the half plane, HOST [H][W/2+1] double, FFT order (ky = 0..H/2-1,-H/2..-1;
 * kx = 0..W/2), unitary scale (|F(0)|^2 = W*H for a normalised frame).  Synchronise the stream.
 * nfs_get_D2d returns NFS_ERR_STATE on a context created with NFS_FLAG_BIN_ONLY. */
NFS_API int nfs_get_D2d(nfs_ctx* ctx, int lag_index, double* out);
NFS_API int nfs_get_I2d(nfs_ctx* ctx, double* out);

/* Variance form of the fluctuation spectrum: V2d(k) = <|F_t(k) - <F(k)>_t|^2>_t, the power
 * of the field's fluctuations in time with the static image (beam, fringes) removed — half the large-lag plateau
 * 2a{T I_s + B} of the difference spectrum of PAPER.md:L23-25, Eq. 1 (for all lags 1..N-1,
 * sum_tau (N - tau) D2d(k,tau) = N^2 V2d(k)).  Built at no extra cost from the sums the lag kernel keeps for I(q).
 *   nfs_get_variance  V_q HOST [n_qbins]: azimuthal mean of V2d over the same |q| bins as D and I (empty bin: 0.0).
 *   nfs_get_V2d       out HOST [H][W/2+1], same layout as nfs_get_I2d.
 * Both synchronise the stream, are non-destructive snapshots, and return NFS_ERR_STATE before the first frame. */
NFS_API int nfs_get_variance(nfs_ctx* ctx, double* V_q);
NFS_API int nfs_get_V2d(nfs_ctx* ctx, double* out);

/* Per-|q| fit of Eq. 1 (<|Delta I_m(q,tau)|^2> = 2a { T I_s [1 - f(q,tau)] + B })
 * to the azimuthally averaged structure function of the frames pushed so far:
 *     D(b,tau) = A_b [1 - exp(-Gamma_b tau)] + C_b,   A = 2a T I_s (signal plateau), C = 2a B (noise floor),
 * with the single-exponential intermediate scattering function f = exp(-Gamma tau) of diffusive fluctuations (the
 * paper does not print its fitting procedure: reading R19 in DESIGN.md).  Unweighted least squares over the lags that
 * have a frame pair; (A, C) by linear least squares for a trial Gamma, Gamma by a scan of 64 log-spaced rates between
 * 1e-3 / tau_max and 1e2 / tau_min refined by 48 golden-section steps — run on the device, one warp per |q| bin,
 * deterministic.  The model-free f follows as 1 - (D - C) / A.
 *   A_q, C_q, Gamma_q, chi2_q  HOST [n_qbins] double (Gamma per frame; chi2 = sum of squared residuals); any may be
 *                              NULL.  Empty bins and fewer than three usable lags give 0.
 * Synchronises the stream; non-destructive. */
NFS_API int nfs_fit_eq1(nfs_ctx* ctx, double* A_q, double* C_q, double* Gamma_q, double* chi2_q);

/* Number of frames pushed so far; ring capacity in frames; bytes of device memory held. */
NFS_API int64_t nfs_num_frames(const nfs_ctx* ctx);
NFS_API int nfs_ring_capacity(const nfs_ctx* ctx);
NFS_API int64_t nfs_device_bytes(const nfs_ctx* ctx);

/*
 * nfs_azimuthal_mean_static — the azimuthal average of step 5 ("azimuthally averaged power spectra";
 * same |q| bins, DC exclusion and Hermitian weights as nfs_finalize) of ONE 2-D spectrum, for callers that are not
 * allowed to allocate device memory.
 *
 * Why it exists.  Everything else in this header works on a context whose buffers nfs_create obtains with cudaMalloc.
 * That is the wrong shape for three kinds of caller: a live acquisition loop, where a cudaMalloc / cudaFree stalls the
 * whole device for an unpredictable time and so nothing on the per-frame path may allocate; a process whose device
 * memory is owned in full by another allocator (a framework's caching pool, an arena sized at start-up, a MIG / MPS
 * share with a hard cap), where a library-side cudaMalloc fails or eats into somebody else's budget; and plug-in
 * code that is handed device pointers and a stream and told to leave the allocator alone.  This call needs no context
 * and calls no cudaMalloc, cudaFree or allocating library routine, ever.  Its working memory is one array compiled into
 * the library (NFS_STATIC_SCRATCH_BYTES, 2.3 MiB) — the price being that every GPU on which the library is loaded
 * carries that array until the process ends, whether or not this call is used.
 *
 *   d_spec2d    DEVICE [H][W/2+1] double, the layout nfs_get_D2d / nfs_get_I2d / nfs_get_V2d return (ky in FFT order,
 *               kx = 0..W/2), 8-byte aligned.  Read only.
 *   W, H        powers of two in [32,4096], W == H (NFS_ERR_UNSUPPORTED otherwise).
 *   n_qbins     1..NFS_STATIC_MAX_QBINS.  More bins than that do not fit the fixed array: the call returns
 *               NFS_ERR_TOO_LARGE and does nothing (use a context, which sizes its own tables).
 *   d_mean_q    DEVICE [n_qbins] double: mean of the spectrum over bin b, counting the mirrored half plane (0.0 for an
 *               empty bin).
 *   d_counts    DEVICE [n_qbins] int64 or NULL: full-plane pixel count of each bin.
 *   cuda_stream a cudaStream_t cast to void* (NULL: the default stream).  Two kernels are enqueued on it and the call
 *               returns without waiting; outputs are valid, and d_spec2d may be changed, once they have run.
 * The device is the one current at the call.  The FIRST call on each device also looks up where the array lives on that
 * device (cudaGetSymbolAddress, which may make the runtime load the library's code onto the GPU): make that first
 * call during set-up, on every device you will use, and before any stream capture is begun.
 * All calls on one device share the one array.  Nothing in it has to be zero beforehand — each call overwrites every
 * slot it later reads, so leftovers of the previous call are harmless — but two calls whose kernels can run at the same
 * time on the same device (different streams, no ordering between them) overwrite each other's partial sums: order
 * them on one stream or with events.  Calls on different devices are independent.
 * Results are deterministic (fixed summation order, no floating-point atomics) and agree with nfs_finalize's binning
 * of the same spectrum to fp64 rounding; bin counts agree exactly.
 * Returns NFS_OK, NFS_ERR_INVALID_ARG (NULL / misaligned pointer, bad size), NFS_ERR_UNSUPPORTED, NFS_ERR_TOO_LARGE, or
 * NFS_ERR_CUDA (no device, launch failure).
 */
#define NFS_STATIC_MAX_QBINS 1024
#define NFS_STATIC_SCRATCH_BYTES (148 * 2 * NFS_STATIC_MAX_QBINS * 8)
NFS_API int nfs_azimuthal_mean_static(const double* d_spec2d, int W, int H, int n_qbins, double* d_mean_q, int64_t* d_counts,
                                      void* cuda_stream);

/* Forget all frames (accumulators, ring, reference, sticky errors); keeps the plan and the memory. */
NFS_API int nfs_reset(nfs_ctx* ctx);
NFS_API void nfs_destroy(nfs_ctx* ctx);
NFS_API const char* nfs_strerror(int status);
/* Text of the first CUDA error seen by this context ("" if none). */
NFS_API const char* nfs_last_cuda_error(const nfs_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* NFS_H_ */
