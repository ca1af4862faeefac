/* fitrig.h -- C ABI of the B200-native FITrig hot path (arxiv 2509.21754).
 *
 * The library computes, on one NVIDIA B200 (sm_100a):
 *   1. the tLISI transient-index map of a time series of radio snapshot images
 *      (Eq. 2-6), one value per N_T x N_T tile and per three-snapshot
 *      unit, and
 *   2. the significance-thresholded, compacted candidate list
 *      (image domain: Eq. 8-9; image-frequency domain: Eq. 10-12,
 *      PAPER.md:343-359 with h = maximum spectral magnitude, or harmonic summing).
 *
 * Citations are /root/reference/PAPER.md line numbers.  "R<n>" are the readings of silent or
 * ambiguous passages listed in DESIGN.md.
 *
 * Conventions
 *   - Snapshots x_0 .. x_{L-1}: H x W fp32, row-major, finite values (R9).  Pixel magnitudes
 *     below the fp32 normal range (|x| < 1.2e-38, other than exact zero) are unsupported.
 *   - Unit u = 0 .. L-3 uses x_u, x_{u+1}, x_{u+2}; x_{u+1} is the reference image
 *     (the paper's s = u + 1).  U = L - 2 units.  (With params.accumulate = g > 1 read
 *     "accumulated snapshot A_j" for x_j and L / g for L throughout.)
 *   - Tiles: Ty = ceil(H / N_T), Tx = ceil(W / N_T); partial edge tiles keep their own pixel
 *     count (R5).  Maps are [U][Ty][Tx], row-major.
 *   - Image axes: x = column (fastest), y = row (R16).
 *   - Every call returns FITRIG_OK (0) or a negative FITRIG_ERR_* code; fitrig_last_error()
 *     then describes it.  No exceptions, no abort, nothing printed.
 *   - There is NO CPU fallback: without a CUDA device every compute call fails with
 *     FITRIG_ERR_CUDA.
 *   - Threads: a context is NOT thread-safe -- it owns one set of workspaces, one current map and two result slots, so
 *     calls on the same context must not overlap (serialise them, or give every thread its own context).  Different
 *     contexts may be used from different threads at the same time, on the same or on different devices; the
 *     library's only shared state is set-up work done once per device under a lock, and fitrig_last_error() is
 *     thread-local.  fitrig_choose_accumulate_static is the exception noted at its declaration (one scratch per device).
 *   - Pointers are marked (device) or (host).  Nothing here is a torch type; a CUDA stream is
 *     passed as void* (cudaStream_t; NULL = the legacy default stream).
 *   - Environment: the library reads these integer DEBUG / TUNING switches, once per fitrig_create (and once per
 *     fitrig_plan_query) call, never later; unset or 0 = the default behaviour.  They change how the work is cut and
 *     launched, never a result (the parity tests run every one of them against the same expected maps):
 *       FITRIG_BOX_TILES=n       fused kernel: n adjacent 32x32 pixel blocks per TMA box (1..8) instead of the planned width
 *       FITRIG_STAGES=n          fused kernel: ring of n boxes per CTA
 *       FITRIG_GRID=n            fused kernel: n CTAs instead of one per SM
 *       FITRIG_EVICT_FIRST=1     fused kernel: L2 evict_first hint on the streaming loads
 *       FITRIG_FORCE_GENERIC=1   take the generic kernel even where the fused TMA kernel applies
 *       FITRIG_OLD_GENERIC=1     generic path: the three-reads-per-pixel kernel instead of the time-marching one
 *       FITRIG_NO_PITCHED_COPY=1 fitrig_stream: one copy per snapshot and strip instead of one pitched copy per strip
 *       FITRIG_NO_PDL=1          plain stream-ordered launches instead of programmatic dependent launches
 *       FITRIG_MARCH_CONS=n      generic kernel: n consumer warps per CTA (default 23 with TMA boxes, 16 with cp.async rows)
 *       FITRIG_MARCH_PROD=n      generic kernel, cp.async variant: n producer warps per CTA (default 8)
 *       FITRIG_MARCH_BOX_KB=n    generic kernel: boxes of about n KB (default 32)
 *       FITRIG_NO_UNALIGNED_FUSED=1  images whose rows do not start on 16-byte boundaries: the generic kernel even where
 *                                the fused kernel's super-row variant applies (cells of 1, 2, 4, 8, 16, 32 pixels)
 *       FITRIG_TEST_FAIL_UNALIGNED_ENCODE=1  behave as if the driver had refused the tensor map of the super-row variant
 *                                (whose rows overlap: accepted by the driver this was built on, not promised by any
 *                                document); the library then takes the generic kernel for that call, as it does when a
 *                                driver really refuses
 */
#ifndef FITRIG_H_
#define FITRIG_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FITRIG_OK 0
#define FITRIG_ERR_INVALID_ARG (-1) /* H,W < 1; L < 3 (R10); tile < 1; NULL pointer; bad strip_rows / mode   */
#define FITRIG_ERR_CUDA (-2)        /* a CUDA call failed; message carries cudaGetErrorString                 */
#define FITRIG_ERR_NOMEM (-3)       /* device or pinned-host allocation failed                                */
#define FITRIG_ERR_STATE (-4)       /* fitrig_detect / getters before any fitrig_tlisi / fitrig_stream        */
#define FITRIG_ERR_CAPACITY (-5)    /* more candidates than `capacity`: first `capacity` written, n_found=all */

#define FITRIG_REF_ABS 0     /* x_hat = |x|, |x| == 0 -> C   (default, R1)                       */
#define FITRIG_REF_LITERAL 1 /* x_hat = x,   x == 0   -> C   (Eq. 5 exactly as printed)          */
#define FITRIG_REF_FLOOR 2   /* x_hat = max(x, C)                                                */

#define FITRIG_BRANCH_IMAGE 0     /* Eq. 8-9   z-score of each unit's tile matrix                  */
#define FITRIG_BRANCH_FREQUENCY 1 /* Eq. 10-12 temporal DFT of each tile's series, h = max |F_k|   */

typedef struct fitrig_ctx fitrig_ctx; /* opaque; owns every workspace and the current map */

/* Zero-initialised == the paper's defaults. */
typedef struct {
  int32_t tile;       /* N_T >= 1; 0 -> 32                                         */
  float C;            /* Eq. 5 constant; <= 0 -> 1e-6; otherwise must be >= 1e-30   */
  int32_t ref_mode;   /* FITRIG_REF_*                                                             */
  float M_override;   /* > 0: use as M instead of the global maximum; 0 -> compute */
  int32_t branch;     /* FITRIG_BRANCH_*                                                          */
  int32_t strip_rows; /* fitrig_stream strip height, multiple of tile; 0 -> auto                  */
  int32_t device;     /* CUDA device ordinal                                                      */
  int32_t row_offset; /* row shards (fitrig_shard_*): image row of this context's first row, a multiple of */
                      /* tile; added to the y of every candidate.  0 for a whole image                     */
  int32_t accumulate; /* g >= 1; 0 -> 1.  Snapshot accumulation (Fig. 16): the images the method  */
                      /* assesses are A_j = x_{gj} + .. + x_{gj+g-1}, j < L / g (an incomplete trailing group  */
                      /* is left out, R25); units U = L / g - 2; M is the largest accumulated pixel          */
  int32_t harmonics;  /* frequency branch: H = 1, 2, 4, .., 32; 0 -> 1.  The spectral refinement h of Eq. 10:          */
                      /* H = 1 maximum magnitude; H > 1 harmonic summing (R26):      */
                      /* eta = max over k and h in {1,2,4..H}, h*k <= U/2, of (|F_k| + |F_2k| + .. + |F_hk|)/sqrt(h) */
  int32_t stride;     /* 0 -> tile.  Window stride in pixels, a divisor of tile.  stride == tile: the paper's         */
                      /* non-overlapping tiles.  stride < tile: OVERLAPPING windows of tile pixels     */
                      /* every stride pixels (an extension, R27); Ty = max(1, ceil(H/stride) - tile/stride + 1);     */
                      /* image branch only, no accumulation, no row shards; candidate (x, y) stays the peak pixel    */
  int32_t batch;      /* B >= 1; 0 -> 1.  B independent stacks of the same shape per call (e.g. the 16 frequency channels of  */
                      /* BASELINE.json configs[4], R19): maps are [B][U][Ty][Tx], statistics and M are per stack, and one    */
                      /* fitrig_detect returns all B candidate lists back to back.  Not with row shards, fitrig_stream,     */
                      /* fitrig_push or overlapping windows                                                               */
  int32_t reserved[4];
} fitrig_params;

/* One candidate, 16 bytes.
 * Image branch:     (x, y) = pixel of max |D^(s) - D^(s+1)| inside the selected tile, first in
 *                   row-major order on ties (R20); the paper's tile index is (y / N_T, x / N_T);
 *                   snapshot = unit index u; score = z_t^(s) of Eq. 8.
 * Frequency branch: (x, y) = tile centre; snapshot = k*, the DFT bin of the spectral maximum
 *                   (frequency k* / (U * T_s)); score = z_t of Eq. 11 (R18). */
typedef struct {
  int32_t x, y, snapshot;
  float score;
} fitrig_candidate;

/* Sub-tile position of a candidate of the frequency branch (fitrig_localise), 24 bytes. */
typedef struct {
  double x, y;  /* pixels; pixel centres at integers, so the centre of tile tx is (tx + 0.5) * N_T - 0.5 */
  double value; /* the interpolated eta surface at (x, y) */
} fitrig_position;

#define FITRIG_INTERP_BILINEAR 0 /* piecewise linear                                                        */
#define FITRIG_INTERP_BICUBIC 1  /* cubic convolution, Keys (1981) a = -1/2, Keys' boundary samples            */
#define FITRIG_INTERP_SPLINE 2   /* cubic spline, not-a-knot end conditions (the scheme of PAPER.md:385)        */
#define FITRIG_INTERP_MAKIMA 3   /* modified Akima piecewise cubic Hermite                                     */

/* How the library will run a problem; pure host arithmetic (no CUDA call), see fitrig_plan_query. */
typedef struct {
  int32_t units, Ty, Tx;     /* map dimensions                                                   */
  int32_t path;              /* 0: fused time-marching kernel (registers): cells of 1, 2, 4, 8, 16 or 32 pixels -- the  */
                             /*    tile itself, a divisor of it (12 = 3 x 4, 48 = 3 x 16, 64 = 2 x 32 ...) or the stride */
                             /*    of overlapping windows.  Rows that do not start on 16-byte boundaries (W % 4 != 0, or */
                             /*    -- known only at the call -- an unaligned stack pointer) ride it through a tensor map */
                             /*    of "super rows" of k = 4 / gcd(W, 4) image rows when the stack's row count is a       */
                             /*    multiple of k and nothing is accumulated; boxes are then at most 7 blocks wide        */
                             /* 1: generic time-marching kernel (shared-memory ring): any other cell size (5, 7, 10 ..), */
                             /*    and whatever the fused kernel cannot take; any width, any alignment                   */
  int32_t units_per_cta;     /* fused path: (box column, unit) pairs per CTA, ceil(boxes * U / grid) */
  int32_t box_tiles;         /* fused path: adjacent 32x32 pixel blocks fetched as one TMA box (1..8) */
  int32_t warps_per_cta;     /* fused path: box_tiles consumer warps + 1 producer warp           */
  int32_t stages;            /* fused path: depth of the CTA's ring of TMA boxes                 */
  int32_t grid;              /* CTAs launched                                                    */
  int32_t smem_bytes;        /* dynamic shared memory per CTA                                    */
  int32_t strip_rows;        /* fitrig_stream: rows per strip (multiple of N_T)                  */
  int32_t n_strips;          /* fitrig_stream: strips per image                                  */
  int32_t n_strip_buffers;   /* fitrig_stream: device strip buffers in rotation                  */
  int32_t reserved;
  int64_t strip_buffer_bytes;
  int64_t workspace_bytes;   /* device bytes fitrig_create allocates (without strip buffers)     */
} fitrig_plan;

/* fitrig_plan_query -- derive tile grid and launch plan for L snapshots of H x W on a device with
 * `num_sms` SMs (0 -> 148, one B200).  Host only; usable without a GPU.  Tile grid per R5.
 * Errors: FITRIG_ERR_INVALID_ARG as for fitrig_create. */
int fitrig_plan_query(int32_t H, int32_t W, int32_t n_snapshots, const fitrig_params* params /*host, may be NULL*/,
                      int32_t num_sms, fitrig_plan* out /*host*/);

/* fitrig_create -- allocate a context for L = n_snapshots images of H x W.
 * params (host) may be NULL (all defaults).  *out receives the context; caller frees it with
 * fitrig_destroy.  Allocates device workspaces proportional to the MAP (U*Ty*Tx), never to the
 * images.  Errors: INVALID_ARG (H, W < 1; L < 3; tile < 1; unknown ref_mode / branch; strip_rows not
 * a multiple of tile), CUDA, NOMEM. */
int fitrig_create(int32_t H, int32_t W, int32_t n_snapshots, const fitrig_params* params, fitrig_ctx** out);

/* fitrig_destroy -- free everything the context owns (synchronises the device).  NULL is OK. */
int fitrig_destroy(fitrig_ctx* ctx);

/* fitrig_map_dims -- U = L - 2 units and the Ty x Tx tile grid.  Any out may be NULL. */
int fitrig_map_dims(const fitrig_ctx* ctx, int32_t* units, int32_t* Ty, int32_t* Tx);

/* fitrig_tlisi -- the tLISI map of a device-resident stack (Eq. 2-6; steps a1-a7 of DESIGN.md).
 *   d_stack (device)  [L][H][W] fp32, contiguous; owned by the caller, read once, never written.  4-byte alignment is
 *                     enough; when d_stack is not 16-byte aligned the fused kernel's loads start at the 16-byte boundary
 *                     below it, i.e. up to 12 bytes BEFORE d_stack are read (and ignored): they must be readable, which
 *                     they are whenever d_stack points into a larger allocation (the only way to get such a pointer).
 *   d_tlisi (device)  [U][Ty][Tx] fp32 tLISI = 1 - q; may be NULL.  Owned by the caller.
 * The context keeps q = 1 - tLISI in fp32 (its complement carries the signal, R21), the per-tile
 * raw sums, the global M and per-unit mean / population std of q (Eq. 8, R3); this
 * "current map" is what fitrig_detect consumes.  Asynchronous on `cuda_stream`.
 * Errors: INVALID_ARG (NULL stack), CUDA. */
int fitrig_tlisi(fitrig_ctx* ctx, const float* d_stack, float* d_tlisi, void* cuda_stream);

/* fitrig_tlisi_batch -- fitrig_tlisi for a context created with params.batch = B > 1 (or 1):
 *   d_stacks (host)   array of B device pointers, each one stack [L][H][W] fp32 as for fitrig_tlisi.
 *   d_tlisi (device)  [B][U][Ty][Tx] or NULL.
 * The B stacks are independent problems (own M, own statistics); the B tLISI kernels run back to back and ONE finalise
 * launch serves all of them.  fitrig_tlisi on such a context reads d_stack as [B][L][H][W].  Errors as fitrig_tlisi. */
int fitrig_tlisi_batch(fitrig_ctx* ctx, const float* const* d_stacks, float* d_tlisi, void* cuda_stream);

/* fitrig_detect -- threshold the current map at z > sigma_threshold (strict, R6) and return the
 * compacted candidate list (Eq. 9, or Eq. 10-12 when params.branch = FREQUENCY).
 *   h_out (host)      room for `capacity` candidates, sorted ascending by (snapshot-or-unit,
 *                     tile row, tile col); frequency branch: by (tile row, tile col).
 *   n_found (host)    total number of candidates (may exceed capacity -> FITRIG_ERR_CAPACITY).
 * May be called repeatedly with different thresholds without recomputing the map.  sigma == 0 for
 * a unit (identical snapshots, one tile) gives z = 0 and no candidate (R4).  Synchronises
 * `cuda_stream` once.  Errors: STATE (no current map), INVALID_ARG, CAPACITY, CUDA. */
int fitrig_detect(fitrig_ctx* ctx, float sigma_threshold, fitrig_candidate* h_out, int64_t capacity,
                  int64_t* n_found, void* cuda_stream);

/* fitrig_detect_batch -- fitrig_detect that also reports how the list divides among the B stacks of the context:
 * h_out holds the candidates of stack 0, then stack 1, ... (each in the order above); n_found_per_stack (host, B
 * entries) receives each stack's total, *n_found their sum.  One compaction launch and one synchronisation for all
 * B stacks. */
int fitrig_detect_batch(fitrig_ctx* ctx, float sigma_threshold, fitrig_candidate* h_out, int64_t capacity,
                        int64_t* n_found, int64_t* n_found_per_stack, void* cuda_stream);

/* fitrig_detect_launch / fitrig_detect_fetch -- fitrig_detect in two halves, for pipelines that keep the device busy
 * while the host reads results: launch enqueues the compaction of the current map on cuda_stream and returns at once;
 * fetch waits for the OLDEST launch that has not been fetched (only for it: work queued behind it keeps running) and
 * delivers its list exactly as fitrig_detect would (h_out needs the capacity given to that launch).  Results live in
 * two slots, so at most two launches may be in flight (a third: FITRIG_ERR_STATE):
 *     tlisi(A); launch;  tlisi(B); launch;  fetch -> A's candidates;  tlisi(C); launch;  fetch -> B's; ...
 * fitrig_detect == launch + fetch (and refuses to run while a launch is unfetched).  n_found_per_stack (host, B
 * entries) may be NULL. */
int fitrig_detect_launch(fitrig_ctx* ctx, float sigma_threshold, int64_t capacity, void* cuda_stream);
int fitrig_detect_fetch(fitrig_ctx* ctx, fitrig_candidate* h_out, int64_t* n_found, int64_t* n_found_per_stack);

/* fitrig_localise -- sub-tile localisation by interpolating the spectrum matrix eta (section 2.4.2:
 * "interpolation methods are activated for precise pulsar localisation in the selected regions ... bilinear, spline,
 * bicubic, or Makima cubic interpolation"; spline interpolation of the spectrum matrix, the peak
 * position is the pulsar position).  The paper names the schemes and prints no rule; reading R28:
 *   - eta_t is a sample of a surface at the centre of tile t; the surface is the tensor product (along x within every
 *     tile row, then along y) of the chosen 1-D scheme on the uniform grid of tile centres (a partial edge tile sits
 *     at its nominal full-tile centre);
 *   - for every candidate the surface is evaluated at x = x_c + i / r, y = y_c + j / r, i, j = -N_T r .. +N_T r
 *     (r = oversample >= 1; (x_c, y_c) the centre of the candidate's tile), without the points outside the hull of
 *     the tile centres, and the position is the largest value, the first in (j, i) row-major order on ties.
 *   h_cands (host)  n candidates as fitrig_detect returned them for the frequency branch ((x, y) inside the tile)
 *   h_eta (host)    NULL: the context's current eta (needs a previous fitrig_detect); otherwise a caller-supplied
 *                   [Ty][Tx] fp32 matrix to interpolate instead (e.g. an eta averaged over several windows)
 *   h_out (host)    n positions
 * Frequency-branch contexts without batch.  Synchronises.  Errors: INVALID_ARG (NULL, method, oversample outside
 * 1..8, a candidate outside the image, image branch, batch), STATE (no eta yet), NOMEM, CUDA. */
int fitrig_localise(fitrig_ctx* ctx, const fitrig_candidate* h_cands, int64_t n, int32_t method, int32_t oversample,
                    const float* h_eta, fitrig_position* h_out, void* cuda_stream);

/* fitrig_stream -- same result as fitrig_tlisi for snapshots that live in HOST memory
 * (Fig. 14: transfers overlapped with the trigger kernels; here at row-strip
 * granularity so images need not be resident).
 *   h_snapshots (host) array of L host pointers, each [H][W] fp32.  Pinned (page-locked) memory
 *                      is needed for the copies to overlap compute; pageable memory works, slowly.
 *   h_tlisi (host)     [U][Ty][Tx] fp32, may be NULL; valid after `cuda_stream` is synchronised.
 * Strips of params.strip_rows rows (all L snapshots of those rows) rotate through device
 * buffers: strip i+1 is copied while strip i is reduced.  Errors: INVALID_ARG, NOMEM, CUDA. */
int fitrig_stream(fitrig_ctx* ctx, const float* const* h_snapshots, float* h_tlisi, void* cuda_stream);

/* Real-time mode ("for real-time processing, this maximum can be estimated from at least
 * three past snapshots"; timeline of Fig. 14: while the n-th tLISI is computed the
 * (n+3)-th snapshot is loaded).  Image branch: the context must have been created with n_snapshots = 3 (one unit
 * per push, maps are [1][Ty][Tx]).  Frequency branch (the image-frequency FITrig IS this streamed
 * computation; reading R29): a context created with n_snapshots = L_w keeps the tLISI cube of the LAST U = L_w - 2
 * units as a ring (map row n mod U holds unit n), every matrix normalised by the running maximum, and once U units
 * exist each push runs Eq. 10-12 over that cube: candidates as for fitrig_detect in the frequency branch
 * (snapshot = k*); before that n_found = 0.  |F_k| does not depend on where the ring starts.
 *
 * fitrig_push -- feed ONE new H x W snapshot (host, pinned for overlap, or device; NULL to flush) and get
 * the result of the unit whose three snapshots had been pushed BEFORE this call:
 *   - the copy of `snapshot` into a device ring of 4 snapshots is started on a private stream, and
 *   - overlapped with it, unit n = x_n, x_{n+1}, x_{n+2} (0-based push order) is computed on
 *     `cuda_stream`: steps a1-a8 with M_n = max(largest pixel of x_0 .. x_{n+2}, C), the running maximum
 *     of everything seen so far (z and therefore the candidates do not depend on M).
 *   *unit (host)    index n of the unit computed by this call, or -1 (the first three pushes; or nothing left)
 *   d_tlisi (device) [Ty][Tx] tLISI of that unit (the newest matrix of the cube), may be NULL
 *   h_out, capacity, n_found  as fitrig_detect; candidate.snapshot = n
 * So push(x_0), push(x_1), push(x_2) return unit = -1; push(x_3) returns unit 0; ...; push(NULL) returns
 * the last unit.  After a call with unit >= 0 the context's current map is that unit's (getters work).
 * The copy is asynchronous: a pushed buffer must stay valid and unchanged until the NEXT fitrig_push that
 * returns a unit >= 0 has returned (or until fitrig_push_reset).  Synchronises `cuda_stream` when a unit
 * is computed.  Errors: INVALID_ARG (image branch without n_snapshots = 3; accumulation; batch; overlapping windows),
 * NOMEM, CUDA, CAPACITY.  (Every tile size works, tiles of 64, 96 .. pixels included: they are merged from 32-pixel cells.)
 *
 * fitrig_push_reset -- forget all pushed snapshots and the running maximum (synchronises the device). */
int fitrig_push(fitrig_ctx* ctx, const float* snapshot, float sigma_threshold, float* d_tlisi,
                fitrig_candidate* h_out, int64_t capacity, int64_t* n_found, int64_t* unit, void* cuda_stream);
int fitrig_push_reset(fitrig_ctx* ctx);

/* Row shards (tiles are independent).  One image is cut into
 * horizontal shards of whole tile rows, one context (normally one GPU) per shard, each created with the
 * shard's own H and params.row_offset.  Only the three global scalars of the method couple the shards:
 * M and, per unit, the mean and standard deviation of the tile matrix (Eq. 8).  Protocol
 * (the frequency branch adds the second exchange described below):
 *     fitrig_tlisi(shard)                       local map, provisional (M of the shard alone)
 *     fitrig_shard_export -> v[2 + 2U]          what the other shards need
 *     all-gather v over the shards              the ONE exchange step (NCCL; (2 + 2U) * 8 bytes per rank)
 *     fitrig_shard_import(all v, world)         global M, mu, sigma; this shard's q and tLISI rescaled
 *     fitrig_detect                             this shard's candidates, y already in image rows
 *
 * fitrig_shard_export -- d_out (device) receives 2 + 2U doubles:
 *   [0]            largest pixel value of this shard's L snapshots (signed, not floored at C; R2)
 *   [1]            number of tiles per unit in this shard
 *   [2 .. 2+U)     per unit: MEAN over this shard's tiles of p = (sum Delta / n_t) * max Delta * (sum r / n_t), i.e.
 *                  the product of Eq. 2 / Eq. 6 WITHOUT the 1/M^2 factor (q = p / M^2)
 *   [2+U .. 2+2U)  per unit: M2 = sum over this shard's tiles of (p - that mean)^2
 * ((n, mean, M2) triples merge without cancellation -- Chan's formula -- so a constant map keeps sigma == 0 exactly, R4.)
 * Asynchronous on cuda_stream.  Errors: STATE (no current map), INVALID_ARG (NULL, batch), CUDA. */
int fitrig_shard_export(fitrig_ctx* ctx, double* d_out, void* cuda_stream);

/* fitrig_shard_import -- d_all (device): `world` export vectors back to back, [world][2 + 2U], in shard
 * order (identical on every shard so that all shards derive bit-identical M, mu, sigma).  Sets
 * M = max(max over shards, C), mu_u and sigma_u of q = p / M^2 over ALL tiles of the image (population
 * std, R3: the shards' (n, mean, M2) merged in shard order, n += n_b, mean += d n_b / n, M2 += M2_b + d^2 n_a n_b / n
 * with d = mean_b - mean_a; mu = mean / M^2, sigma = sqrt(M2 / n) / M^2), rewrites this shard's q and tLISI with
 * that M, and writes tLISI to d_tlisi (device,
 * [U][Ty_shard][Tx], may be NULL).  The shard's map is then bit-identical to the same rows of a
 * whole-image fitrig_tlisi.  Asynchronous.  Errors: STATE, INVALID_ARG (NULL, world < 1), CUDA. */
int fitrig_shard_import(fitrig_ctx* ctx, const double* d_all, int32_t world, float* d_tlisi, void* cuda_stream);

/* Row shards, frequency branch: eta (Eq. 10) scales with 1 / M^2, so it can only be formed after the first exchange,
 * and the z-score of Eq. 11 runs over the eta of ALL tiles of the image: a second, 3-double exchange.
 *     ... fitrig_shard_import as above ...
 *     fitrig_shard_export_eta -> w[3]           eta and k* of this shard's tiles; w = (tiles, mean eta, sum (eta - mean)^2)
 *     all-gather w over the shards
 *     fitrig_shard_import_eta(all w, world)     global mean and population std of eta (Chan's merge in shard order)
 *     fitrig_detect                             Eq. 12 on this shard's tiles
 * Both are asynchronous on cuda_stream.  Errors: STATE (no map / export_eta not called), INVALID_ARG (NULL, image
 * branch, batch), CUDA. */
int fitrig_shard_export_eta(fitrig_ctx* ctx, double* d_out /*device, 3 doubles*/, void* cuda_stream);
int fitrig_shard_import_eta(fitrig_ctx* ctx, const double* d_all /*device, [world][3]*/, int32_t world, void* cuda_stream);

/* fitrig_choose_accumulate -- the stopping rule of snapshot accumulation (section 3.3.2: "Snapshots can be
 * combined progressively until there is enough difference between adjacent accumulated snapshots").  The paper gives
 * neither the measure nor the threshold; reading R30: the group sizes g = 1, 2, 4, .., 32 with g <= g_max and
 * at least 3 accumulated snapshots left are tried in this order (Fig. 16's pairwise tree), and the first
 * whose contrast
 *     d(g) = mean over j, pixels of |A_{j+1} - A_j|  /  mean over j, pixels of |A_j|,   A_j = x_{gj} + .. + x_{gj+g-1}
 * (the difference image of Eq. 3 on accumulated snapshots over the intensity level Eq. 4 normalises by) reaches eps
 * (d >= eps) is returned; if none does, the largest admissible g.  The result goes into fitrig_params.accumulate.
 *   d_stack (device)  [n_snapshots][H][W] fp32, contiguous; read once per level tried
 *   g_out (host)      the group size
 *   contrast (host)   d of the levels looked at, g = 1, 2, 4, .. up to the returned one (room for 6); may be NULL
 *   n_levels (host)   how many that is; may be NULL
 * Needs no context.  Synchronises cuda_stream.  Errors: INVALID_ARG (NULL, H, W < 1, n_snapshots < 3, g_max < 1, eps NaN,
 * device), NOMEM, CUDA. */
int fitrig_choose_accumulate(const float* d_stack, int32_t H, int32_t W, int32_t n_snapshots, float eps, int32_t g_max,
                             int32_t device, int32_t* g_out, double* contrast, int32_t* n_levels, void* cuda_stream);

/* fitrig_choose_accumulate_static -- fitrig_choose_accumulate for callers that must not allocate device memory.
 *
 * Who that is: fitrig_choose_accumulate does two cudaMalloc and two cudaFree on every call.  cudaFree waits until
 * everything queued on the device has drained and cudaMalloc can block for milliseconds behind the driver's locks, so
 * inside the real-time loop (fitrig_push, Fig. 14) they would break the overlap of the next snapshot's copy with the
 * current unit's kernels; and a process whose device memory already belongs to someone else's pool (a framework's
 * caching allocator that has taken the whole card, a fixed per-process memory budget) may simply be refused the
 * allocation.  This entry point calls no cudaMalloc, cudaFree, cudaHostAlloc or any other allocating
 * routine: its scratch (the per-block partial sums of every level and the decision record) is a fixed device array
 * compiled into the library.
 *
 * Arguments, rule, outputs and results are those of fitrig_choose_accumulate (same kernels, same grid, same summation
 * order: the contrasts are bit-identical).  What differs:
 *   - Size limit.  The scratch holds FITRIG_STATIC_ACCUM_MAX_PARTIALS partial sums (128 KB); a call needs
 *     levels * min(ceil(H * W / 256), 8 * SM count) of them, levels = the admissible group sizes g = 1, 2, 4, .. (at
 *     most 6).  On one B200 (148 SMs) the largest request is 6 * 1184 = 7104, so every image size fits there; a request
 *     beyond the limit (a device with more SMs and many levels) is refused with FITRIG_ERR_INVALID_ARG and a message
 *     that gives both numbers -- nothing is launched, nothing is truncated.
 *   - Cost of the array.  Every CUDA device on which the library is loaded holds its own copy of it from load until
 *     the process exits, whether or not this function is ever called.
 *   - First call on a device.  It looks up where that device keeps the array (cudaGetSymbolAddress, which may make
 *     the runtime load the library's kernels onto the device) and the device's SM count, and caches both.  Make that
 *     first call at set-up time, before any stream capture is begun on the device; later calls do no such work.
 *   - One array for everybody.  All calls on a device, from any thread and on any stream, use the same scratch, and
 *     it keeps whatever the last call left in it.  The call clears the decision record itself before it launches (the
 *     partial sums are all rewritten before they are read), so calls issued one after the other need no care; two
 *     calls whose GPU work OVERLAPS (two host threads, each with its own stream) race on the array and may both return
 *     wrong results.  Serialise them, or give all but one fitrig_choose_accumulate.
 * Synchronises cuda_stream, like fitrig_choose_accumulate.  Errors: INVALID_ARG (as fitrig_choose_accumulate; the size
 * limit; device ordinal >= 64), CUDA. */
#define FITRIG_STATIC_ACCUM_MAX_PARTIALS 8192
int fitrig_choose_accumulate_static(const float* d_stack, int32_t H, int32_t W, int32_t n_snapshots, float eps,
                                    int32_t g_max, int32_t device, int32_t* g_out, double* contrast, int32_t* n_levels,
                                    void* cuda_stream);

/* fitrig_get_stats -- M (B floats) and the per-unit mean / population std of q = 1 - tLISI
 * (Eq. 8; mu_tLISI = 1 - mu_q; B * U doubles each, row b * U + u).  Frequency branch after fitrig_detect: entry
 * b * U of mu and sigma (unit 0 of stack b) describes eta of that stack (Eq. 11) instead.  Host outputs, each may
 * be NULL.  Synchronises. */
int fitrig_get_stats(const fitrig_ctx* ctx, float* M, double* mu, double* sigma);

/* fitrig_get_map -- copy one of the context's maps to host memory (synchronises).
 *   which = 0: q = 1 - tLISI   [B][U][Ty][Tx] fp32   which = 1: tLISI        [B][U][Ty][Tx] fp32
 *   which = 2: eta (Eq. 10)    [B][Ty][Tx] fp32      which = 3: k* as fp32   [B][Ty][Tx]
 * 2 and 3 need the frequency branch and a previous fitrig_detect. */
int fitrig_get_map(const fitrig_ctx* ctx, int32_t which, float* h_out);

/* fitrig_get_raw -- per-tile partial results of Eq. 6, each [B][U][Ty][Tx], host, may be
 * NULL: sum of Delta, max of Delta, sum of r, and the first max-Delta pixel as x and y (R20). */
int fitrig_get_raw(const fitrig_ctx* ctx, float* sumD, float* maxD, float* sumR, int32_t* arg_x, int32_t* arg_y);

/* fitrig_profile -- enable (1) / disable (0) CUDA-event timing of the library's own kernels on the
 * launching stream; either call starts a new accumulation window.  fitrig_last_timing then reports, for all
 * fitrig_tlisi / fitrig_stream calls since the window started, the summed duration of the fused (or generic)
 * tLISI kernel launches and their number, and the summed duration and number of the finalise+statistics
 * launches, in milliseconds (synchronises the device), and starts a new window.  Any out may be NULL. */
int fitrig_profile(fitrig_ctx* ctx, int32_t enable);
int fitrig_last_timing(const fitrig_ctx* ctx, float* main_kernel_ms, int32_t* main_kernel_launches,
                       float* finalize_ms, int32_t* finalize_launches);

/* fitrig_probe_read_bandwidth -- calibration for roofline figures: the best rate (GB/s) at which a plain read-only
 * kernel (coalesced 16-byte loads, no arithmetic to speak of) streams `bytes` bytes of d_buf (device, 16-byte
 * aligned) in `reps` timed passes on this device.  Synchronises.  Not part of the method. */
int fitrig_probe_read_bandwidth(fitrig_ctx* ctx, const void* d_buf, int64_t bytes, int32_t reps, float* gbs,
                                void* cuda_stream);

/* fitrig_stream_timeline -- the copy / compute timeline of the last fitrig_stream that ran with fitrig_profile(1)
 * (Fig. 13-14: the transfer of the next input overlapped with the trigger kernel of the current one;
 * here per row strip).  ms (host) receives, for each of the first `capacity` strips, four times in milliseconds
 * relative to the start of the first copy: copy start, copy end (on the library's copy stream), kernel start, kernel
 * end (on the caller's stream); *n_strips the number of strips of that call.  Synchronises.  Errors: STATE. */
int fitrig_stream_timeline(const fitrig_ctx* ctx, float* ms, int32_t capacity, int32_t* n_strips);

/* fitrig_launch_count -- kernels launched by this context since creation (for bench.py's gpu_launches). */
int fitrig_launch_count(const fitrig_ctx* ctx, int64_t* n);

/* fitrig_copy_count -- host-to-device copy calls issued by this context's fitrig_stream / fitrig_push since creation
 * (one per strip when the snapshots travel as pitched copies, L per strip otherwise; one per pushed snapshot). */
int fitrig_copy_count(const fitrig_ctx* ctx, int64_t* n);

/* fitrig_last_error -- thread-local message of the last failing call on this thread; never NULL. */
const char* fitrig_last_error(void);

/* fitrig_version -- "fitrig-b200 <major>.<minor>". */
const char* fitrig_version(void);

#ifdef __cplusplus
}
#endif
#endif /* FITRIG_H_ */
