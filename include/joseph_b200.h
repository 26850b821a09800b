/*
 * joseph_b200.h -- C ABI of libjoseph_b200.so: Joseph's ray-driven 3-D forward projection and its
 * exact adjoint for PET on one NVIDIA B200 (sm_100a), non-TOF and TOF, sinogram and listmode, plus a
 * listmode OSEM driver.  After arxiv 2212.12519 ("parallelproj"); citations are PAPER.md:<line>.
 *
 * The calls follow the paper's problem statement (section 2.2): the low-level
 * projectors take "a list of coordinates representing the start and end point of the rays", are
 * agnostic to scanner geometry, exist in non-TOF and TOF mode, with TOF sinogram ("all available TOF
 * bins along a ray") and TOF listmode ("one specific TOF bin") variants, and the back projections are
 * "the exact adjoint of the forward projections".
 *
 * Conventions (readings A1-A14 are listed in DESIGN.md)
 *   image   f[i0][i1][i2], float32, C order, axis 2 fastest.  n = dims, voxsize v (mm), origin o =
 *           world coordinate (mm) of the CENTRE of voxel [0][0][0].
 *   LOR j   runs from s_j = (xs,ys,zs)[j] to e_j = (xe,ye,ze)[j] (world mm), float32, SoA.
 *   Joseph principal axis p = argmax_a |e_a - s_a| (ties: lowest a, decided on the
 *           exact differences); for every voxel-centre plane x_p = o_p + i v_p crossed by the closed
 *           segment [s,e]: bilinear interpolation of the four nearest neighbours of the crossing
 *           point (voxels outside the image count as zero); sum over planes times
 *           cf = v_p |e-s| / |e_p - s_p|.  A zero-length LOR projects to 0.
 *   TOF one weight per crossed plane, evaluated at the crossing point, whose
 *           signed distance from the LOR midpoint (positive towards e) is tau:
 *             w(tau,c) = 1/2 [ erf(clamp(c+W/2-tau, -m, m)/(sigma sqrt2))
 *                            - erf(clamp(c-W/2-tau, -m, m)/(sigma sqrt2)) ],  m = n_sigmas*sigma,
 *           W = tofbin_width, c = centre of the TOF bin: a Gaussian truncated at +-n_sigmas sigma,
 *           integrated over the bin, not renormalised.  Sinogram bin k = 0..n_tofbins-1 has
 *           c_k = (k - (n_tofbins-1)/2) W + center_offset; listmode bin `it` (signed int16) has
 *           c = it*W + center_offset.
 *
 * Memory   Unless a name ends in _host, ALL data pointers are DEVICE pointers owned by the caller
 *           (e.g. torch tensors); jp_geom / jp_tof / jp_lors structs themselves are read on the host
 *           at call time.  Inputs are const.  The library does not dereference caller pointers after a
 *           call returns, except inside a jp_plan (which owns only its own device buffers).  The library keeps no
 *           state between calls other than the plans the caller creates and destroys.
 * Streams  Every call is asynchronous on the CUDA stream `stream` (a cudaStream_t passed as void*,
 *           NULL = legacy default stream) and never synchronises the device, except the _host calls,
 *           which return after their result is in host memory.
 * Scratch  Some calls use stream-ordered scratch (cudaMallocAsync/cudaFreeAsync on `stream`).
 * Errors   Return 0 on success.  Negative = error, nothing (more) enqueued:
 *             JP_ERR_POINTER (-1) null pointer where data is required
 *             JP_ERR_SIZE    (-2) n < 0, a dim <= 0, voxsize <= 0, n_tofbins < 1 (or > JP_MAX_TOFBINS),
 *                                 sigma <= 0, tofbin_width <= 0, n_sigmas <= 0, n_subsets < 1 ...
 *             JP_ERR_CUDA    (-3) a CUDA runtime call failed; text via jp_last_error()
 *             JP_ERR_PLAN    (-4) invalid plan handle
 *           n == 0 LORs is a successful no-op.  No exceptions or C++ types cross this boundary.
 */
#ifndef JOSEPH_B200_H
#define JOSEPH_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define JP_OK 0
#define JP_ERR_POINTER (-1)
#define JP_ERR_SIZE (-2)
#define JP_ERR_CUDA (-3)
#define JP_ERR_PLAN (-4)

#define JP_MAX_TOFBINS 64

/* image geometry shared by all calls (host struct) */
typedef struct jp_geom {
    int32_t n[3];     /* voxels along axes 0,1,2 (axis 2 fastest in memory) */
    float origin[3];  /* world mm of the centre of voxel [0][0][0] */
    float voxsize[3]; /* mm, > 0, may be anisotropic */
} jp_geom;

/* TOF parameters (host struct), all lengths in mm (x = c t / 2) */
typedef struct jp_tof {
    float tofbin_width_mm;  /* W  > 0 */
    float sigma_tof_mm;     /* sigma > 0 (FWHM / 2.3548) */
    float n_sigmas;         /* truncation, PAPER.md:78 uses 3 */
    int32_t n_tofbins;      /* sinogram bins per LOR (ignored by the listmode calls) */
    float center_offset_mm; /* shift of the bin centres along the LOR, normally 0 */
} jp_tof;

/* LOR end points, struct of arrays, float32, world mm; each array has n elements (device) */
typedef struct jp_lors {
    const float *xs, *ys, *zs; /* start points */
    const float *xe, *ye, *ze; /* end points */
    int64_t n;
} jp_lors;

/* ---- non-TOF ---------------------------------------------------------------------- */
/* p[j] = line integral of img along LOR j.  OVERWRITES p[0..n).  img: n[0]*n[1]*n[2] floats. */
int jp_fwd(const jp_lors *lors, const float *img, const jp_geom *geom, float *p, void *stream);
/* img += A^T y, the exact adjoint of jp_fwd (atomic adds PAPER.md:46).
   ACCUMULATES into img (the caller zeroes it when a plain back projection is wanted).
   Non-finite y: Inf / NaN on a LOR that crosses the image propagate into the voxels of that LOR exactly as a plain
   atomicAdd of cf y w would (track tiles that hold such a value take the per-LOR float path); y of LORs that miss
   the image is never used.  Tracks are staged in shared memory in int32 fixed point with ONE scale per staged
   group of LORs, S = lim / max |cf y| over the group, lim = min(2^22 - 2, 2^31 / (2 L) - 1) for a group of up to L LORs:
     unplanned calls (tiles of 768 consecutive LORs, L = 768):      quantum max|cf y| / lim = 7.2e-7 x the tile's max;
     planned calls (whole track pieces, L = 768 / 1536 / 2304):      7.2e-7 / 1.4e-6 / 2.1e-6 x the track piece's max
     (2304 = the 48 x 48 ring pairs of the paper's scanner).
   Every contribution cf y w is rounded to the nearest multiple of the quantum (error <= half of it); one below half
   a quantum is dropped.  On configs[1] the image error is 2.6e-6 of its maximum (profiles/r02b_parity.txt). */
int jp_back(const jp_lors *lors, const float *y, const jp_geom *geom, float *img, void *stream);

/* ---- TOF sinogram: all n_tofbins bins of every LOR ------------------------------ */
/* p[j*n_tofbins + k], bin fastest.  OVERWRITES p. */
int jp_fwd_tof_sino(const jp_lors *lors, const float *img, const jp_geom *geom, const jp_tof *tof,
                    float *p, void *stream);
/* img += A_tof^T y, y[j*n_tofbins + k].  ACCUMULATES. */
int jp_back_tof_sino(const jp_lors *lors, const float *y, const jp_geom *geom, const jp_tof *tof,
                     float *img, void *stream);

/* ---- TOF listmode: only the TOF bin tofbin[j] of event j --------------------------- */
int jp_fwd_tof_lm(const jp_lors *lors, const int16_t *tofbin, const float *img, const jp_geom *geom,
                  const jp_tof *tof, float *p, void *stream);
int jp_back_tof_lm(const jp_lors *lors, const int16_t *tofbin, const float *y, const jp_geom *geom,
                   const jp_tof *tof, float *img, void *stream);

/* ---- diagnostics --------------------------------------------------------------------------------- */
/* principal_axis[j] in {0,1,2} ("principal direction"); bit-exact against the oracle. */
int jp_classify(const jp_lors *lors, uint8_t *principal_axis, void *stream);

/* total[0] += number of (LOR, plane) pairs the projectors visit for these LORs: planes of the principal
   axis crossed by the closed segment whose crossing point has at least one of its four neighbours
   inside the image (the "plane-steps" the roofline is quoted in).  total: device uint64, caller-zeroed. */
int jp_plane_steps(const jp_lors *lors, const jp_geom *geom, unsigned long long *total, void *stream);
/* the same count for the TOF listmode projectors ("only affected by a few voxels"): only
   the planes whose crossing point lies inside the truncated TOF kernel of the event's own bin,
   |tau - c| <= n_sigmas sigma + W/2, are visited. */
int jp_plane_steps_tof_lm(const jp_lors *lors, const int16_t *tofbin, const jp_geom *geom, const jp_tof *tof,
                          unsigned long long *total, void *stream);

/* ---- listmode OSEM (Hudson & Larkin, PAPER.md:193 ref. 39) ------------------- */
/* n_iter iterations over n_subsets subsets, subset m = events {e : e mod n_subsets == m}, in order:
 *   ybar_e = (A_tof x)_e;  r_e = 1/ybar_e if ybar_e > 1e-9 else 0;  b = A_m^T r;
 *   x <- x * b * n_subsets / sens  where sens > 0, else 0.
 * img: in = start image, out = result.  sens: sensitivity image (device).  workspace: device buffer of
 * at least jp_lm_osem_workspace_bytes() bytes.  All on `stream`, no host synchronisation. */
size_t jp_lm_osem_workspace_bytes(int64_t n_events, const jp_geom *geom, int n_subsets);
int jp_lm_osem(const jp_lors *events, const int16_t *tofbin, const jp_geom *geom, const jp_tof *tof,
               const float *sens, float *img, int n_subsets, int n_iter, void *workspace,
               size_t workspace_bytes, void *stream);

/* ---- listmode plan: sorted events (set-up; BASELINE.json north_star (b)) ---------------- */
/* Listmode events arrive in acquisition order, which makes the image access of the projectors random
 * (PAPER.md:88); the paper names pre-sorting the events as the remedy.  A plan is that
 * sort, done once per event list: the events of every OSEM subset (subset m = {e : e mod n_subsets == m},
 * the rule of jp_lm_osem) are ordered by principal axis, transaxial line, plane and axial position of
 * their TOF bin, and a sorted copy of the end points / TOF bins is kept on the device together with the
 * permutation.  Planned calls compute the projections the unplanned calls compute (path 2 with the same
 * arithmetic per event, the other paths within float32 rounding: other TOF weight table, other order of
 * the floating-point sums) and take / return per-event arrays in CALLER order.
 *   events, tofbin: device arrays, only read during jp_lm_plan_create (not kept).
 *   The plan owns its device buffers (26 + 4 bytes per event) until jp_lm_plan_destroy.  When the sorted events do NOT
 *   come in long runs on one transaxial line (an OSEM subset of a clinical acquisition: ~20 events per line), the plan
 *   also cuts every event into PIECES per image brick of 32 x 32 x 16 cells (csrc/jp_brick.cu; about 3.5 pieces of
 *   32 bytes per event + 8 bytes per event), so that the forward projection can run on bricks held in shared memory
 *   (if the device has no room for the pieces the plan is made without them and the planned calls use path 2).
 *   jp_lm_plan_create allocates with cudaMalloc and SYNCHRONISES `stream` (it reads the per-subset / per-axis event
 *   counts, the run statistics and the piece counts back to the host); the planned calls are asynchronous.  A plan keeps
 *   image-sized scratch (quad image and accumulators, allocated with cudaMalloc on the first call that needs them)
 *   that the planned calls write: use a plan from ONE stream at a time.
 *   n_subsets in 1..255, fewer than 2^31 events.  subset = -1 in the calls below means all events. */
typedef struct jp_plan jp_plan;
int jp_lm_plan_create(const jp_lors *events, const int16_t *tofbin, const jp_geom *geom, const jp_tof *tof,
                      int n_subsets, void *stream, jp_plan **plan);
int jp_lm_plan_destroy(jp_plan *plan);
/* Which kernels the planned listmode projectors and the planned OSEM use:
 *   0  chosen from the plan's run statistics (default): line tiles when the sorted events come in runs of >= 512 on one
 *      transaxial line, else path 3 when the plan could build its brick pieces, else path 2;
 *   1  line tiles (csrc/jp_lm_tile.cu): rows shared by the events of a line, adjoint staged in fixed point per run;
 *   2  quad image (csrc/jp_quad.cu): one 128-bit gather / float atomic add per event and plane;
 *   3  image bricks for the forward projection (csrc/jp_brick.cu: TMA box loads into shared memory), float atomic adds
 *      on the quad accumulators for the adjoint -- the same floating-point semantics as path 2;
 * All paths compute the same projections (tests force each of them); images or TOF kernels a path cannot hold fall
 * back towards path 2.  Path 3 builds the brick pieces if the plan has none (allocates, synchronises).  Not to be
 * changed while a call that uses the plan is being issued from another thread. */
int jp_lm_plan_set_path(jp_plan *plan, int path);
/* number of events of a subset (subset = -1: all); -1 for an invalid plan or subset */
int64_t jp_lm_plan_subset_count(const jp_plan *plan, int subset);
/* p[e] for the events e of the subset (other entries of p are left untouched); p has n entries */
int jp_fwd_tof_lm_planned(const jp_plan *plan, int subset, const float *img, float *p, void *stream);
/* img += A_subset^T y, y has n entries in caller order.  ACCUMULATES. */
int jp_back_tof_lm_planned(const jp_plan *plan, int subset, const float *y, float *img, void *stream);
/* The same projections with the per-event arrays in PLAN order ("pre-sorted" listmode events): entry k
 * of p_sorted / y_sorted belongs to the event at position k of the plan's sorted list, i.e. caller event perm[k].  The
 * planned calls above gather / scatter through the permutation on every call (one 32-byte sector per 4-byte value);
 * callers that project a list many times (OSEM) permute once with jp_lm_plan_permute and use these.
 * jp_lm_plan_permute: to_plan_order != 0: out[k] = in[perm[k]]; else out[perm[k]] = in[k].  in != out, n floats. */
int jp_fwd_tof_lm_planned_sorted(const jp_plan *plan, int subset, const float *img, float *p_sorted, void *stream);
int jp_back_tof_lm_planned_sorted(const jp_plan *plan, int subset, const float *y_sorted, float *img, void *stream);
int jp_lm_plan_permute(const jp_plan *plan, const float *in, float *out, int to_plan_order, void *stream);
/* jp_lm_osem on the plan's events, subsets and geometry */
/* NON-TOF projections of the plan's events (the paper's second listmode workload: every plane
 * of each event's LOR, the TOF bins of the plan are ignored).  Arguments, order of results (caller order) and
 * subset selection as for jp_fwd_tof_lm_planned / jp_back_tof_lm_planned; jp_back_lm_planned ACCUMULATES. */
int jp_fwd_lm_planned(const jp_plan *plan, int subset, const float *img, float *p, void *stream);
int jp_back_lm_planned(const jp_plan *plan, int subset, const float *y, float *img, void *stream);

size_t jp_lm_osem_planned_workspace_bytes(const jp_plan *plan);
int jp_lm_osem_planned(const jp_plan *plan, const float *sens, float *img, int n_iter, void *workspace,
                       size_t workspace_bytes, void *stream);

/* ---- the two halves of one listmode OSEM subset update (multi-GPU) ---------------------------- */
/* Events are independent units: every GPU holds a plan over its own shard of the event list (shards that start at
 * a multiple of n_subsets keep "subset = e mod n_subsets") and the whole image.  Per subset each GPU computes
 *     b = A_m^T r,  r_e = 1/(A x)_e if (A x)_e > 1e-9 else 0        (jp_lm_osem_planned_backratio, OVERWRITES b)
 * over its events, the caller sums b over the GPUs (one all-reduce of n0*n1*n2 floats, the only exchange step),
 * and every GPU applies   x <- x b scale / sens  where sens > 0, else 0;  b <- 0    (jp_osem_update).
 * With one GPU the pair is jp_lm_osem_planned's subset update.  workspace as for jp_lm_osem_planned. */
int jp_lm_osem_planned_backratio(const jp_plan *plan, int subset, const float *x, float *b, void *workspace,
                                 size_t workspace_bytes, void *stream);
int jp_osem_update(float *x, float *b, const float *sens, float scale, const jp_geom *geom, void *stream);

/* ---- image-based resolution model -------------------------------- */
/* out = G in: 3-D Gaussian of standard deviation sigma_mm (mm; FWHM = 2 sqrt(2 ln 2) sigma; the paper uses
 * 4.5 mm FWHM), taps exp(-(k v_a)^2 / (2 sigma^2)) for |k| <= ceil(n_sigmas sigma / v_a), normalised per axis,
 * zero outside the image (so G is symmetric: the same call serves "before forward" and "after back").
 * in / out: device, geom->n voxels, C order; in may equal out.  Asynchronous on `stream`; scratch is
 * stream-ordered.  JP_ERR_SIZE: sigma_mm <= 0, n_sigmas <= 0 or a kernel radius > 16 voxels. */
int jp_gauss3d(const float *in, float *out, const jp_geom *geom, float sigma_mm, float n_sigmas, void *stream);

/* jp_gauss3d for callers that cannot allocate device memory: same arguments, same kernels, bit-identical result,
 * and NO cudaMalloc / cudaMallocAsync / cudaFree (or any allocating library routine) anywhere in the call.
 * Meant for code that runs after all device memory has been handed out (a reconstruction service whose pools were
 * sized at start-up, a framework that owns the whole GPU), for host threads that may not take the allocator's
 * device-wide lock or its implicit synchronisation (acquisition / real-time loops), and for set-ups where the
 * stream-ordered allocator that jp_gauss3d relies on is not available.
 *   Scratch   the image-sized intermediate of the separable passes lives in a fixed array inside the library's own
 *             device data: JP_GAUSS3D_STATIC_MAX_VOXELS floats = 16 MiB, held by every GPU that loads the library
 *             until the process exits.  An image with more voxels than that is refused: JP_ERR_SIZE, text via
 *             jp_last_error(), nothing enqueued.  (200 x 200 x 96, the paper's image, has 3.84 M voxels.)
 *   Set-up    the FIRST call on each device looks up that device's address of the array (cudaGetSymbolAddress,
 *             with the calling thread's current device, which must be the device of `stream`, `in` and `out`);
 *             later calls on that device reuse it.  Make this first call outside any stream capture.
 *   Sharing   all calls on one device use the same array.  Calls on one stream are ordered and safe; two calls
 *             that may overlap on the GPU (different streams, or different host threads on different streams) RACE
 *             on it and give garbage -- order them with events or use jp_gauss3d for one of them.  Nothing needs
 *             clearing between calls: every pass overwrites its whole destination before it is read.
 * in / out: device, caller-owned, geom->n voxels, C order; in may equal out.
 * Errors as for jp_gauss3d. */
#define JP_GAUSS3D_STATIC_MAX_VOXELS 4194304
int jp_gauss3d_static(const float *in, float *out, const jp_geom *geom, float sigma_mm, float n_sigmas, void *stream);

/* jp_lm_osem_planned with the resolution model in every subset (reading R3): ybar = A (G x), b = G (A^T r),
 * x <- x b n_subsets / sens; `sens` is the caller's (it should hold G A^T 1).  Workspace as for
 * jp_lm_osem_planned. */
int jp_lm_osem_planned_res(const jp_plan *plan, const float *sens, float *img, int n_iter, float res_sigma_mm,
                           float res_n_sigmas, void *workspace, size_t workspace_bytes, void *stream);

/* ---- TOF sinogram OSEM with multiplicative factors and additive contamination -------- */
/* PAPER.md:80 ("the projection work required for an OSEM subset update"), :118 (sinogram OSEM keeps "the complete
 * image volume, the emission sinogram, the forward projection and the contamination sinogram" on the GPU).  Model
 *     ybar[j][k] = mult[j] (A x)[j][k] + contam[j][k]
 * (mult: attenuation x normalisation per LOR; contam: randoms + scatter per LOR and TOF bin).  Readings S1-S3:
 *   S1  subset m = LORs [subset_offsets[m], subset_offsets[m+1]) of `lors` (the caller arranges the list subset-major,
 *       e.g. every n_subsets-th view of a ring scanner), m = 0..n_subsets-1 in order;
 *   S2  r[j][k] = mult[j] y[j][k] / ybar[j][k]  if ybar[j][k] > 1e-9 else 0;
 *   S3  x <- x (A_m^T r) / sens_m  where sens_m > 0, else 0;   sens_m = A_m^T (mult (x) 1_bins).
 * subset_offsets: HOST array of n_subsets + 1 non-decreasing offsets in [0, lors->n].  y, contam: device,
 * [lors->n][n_tofbins]; mult: device [lors->n]; mult or contam may be NULL (= 1, = 0).  sens: device
 * [n_subsets][n0*n1*n2].  img: in = start image, out = result.  workspace: device, at least
 * jp_sino_osem_tof_workspace_bytes() bytes (the ratio sinogram of the largest subset; only used when the TOF kernel is
 * wider than the fused kernel supports -- otherwise forward, ratio and back of a subset run as one kernel and the
 * ratio never leaves the chip).  Everything is asynchronous on `stream`, no host synchronisation. */
size_t jp_sino_osem_tof_workspace_bytes(const int64_t *subset_offsets, int n_subsets, int64_t n, const jp_tof *tof);
/* sens[m] = A_m^T (mult (x) 1_bins) for every subset; OVERWRITES sens.  workspace may be NULL unless the TOF
 * kernel is wider than the fused kernels support (then as for jp_sino_osem_tof). */
int jp_sino_sens_tof(const jp_lors *lors, const int64_t *subset_offsets, int n_subsets, const float *mult,
                     const jp_geom *geom, const jp_tof *tof, float *sens, void *workspace, size_t workspace_bytes,
                     void *stream);
int jp_sino_osem_tof(const jp_lors *lors, const int64_t *subset_offsets, int n_subsets, const float *y,
                     const float *mult, const float *contam, const float *sens, const jp_geom *geom, const jp_tof *tof,
                     float *img, int n_iter, void *workspace, size_t workspace_bytes, void *stream);

/* ---- sinogram plan: the structure of a LOR list, found once (set-up; BASELINE.json north_star (b)) ------------------ */
/* The projectors take plain lists of LOR end points.  The lists a ring scanner produces are regular: a
 * sinogram is K TRACKS (runs of LORs with bit-identical transaxial end points xs, ys, xe, ye: the ring pairs of one
 * (view, radial) bin) of T LORs each, and every track has the same axial pattern (zs, ze)[T].  jp_sino_plan_create
 * detects exactly that from the data (T = length of the first run; n a multiple of T; every block of T LORs a track
 * with the pattern of the first) and then keeps 16 bytes per TRACK, the pattern, and a lane order (LORs of a track
 * sorted by |ze - zs|: equal tilt = equal LOR length = identical TOF weights on every plane).  Any other list is kept
 * as a plain copy (24 bytes per LOR) and the planned calls run the kernels of the unplanned calls on it.
 *   lors: device arrays, only read during jp_sino_plan_create (not kept).  The plan is independent of the image
 *   geometry and of the TOF parameters.  jp_sino_plan_create SYNCHRONISES `stream` (it reads the track length and the
 *   regularity flag back) and allocates the plan's device buffers with cudaMalloc; destroy with jp_plan_destroy.
 * Planned calls compute what the unplanned calls compute (same arithmetic per LOR and plane; only the order of the
 * floating-point sums of the back projection differs), take / return per-LOR arrays in CALLER (list) order, are
 * asynchronous on `stream` and use only stream-ordered scratch.  A plan may be used from several streams at once
 * (it is read-only after creation). */
int jp_sino_plan_create(const jp_lors *lors, void *stream, jp_plan **plan);
/* n_lors; n_tracks and track_length (both 0 for a list that is not regular); any output pointer may be NULL */
int jp_sino_plan_info(const jp_plan *plan, int64_t *n_lors, int64_t *n_tracks, int32_t *track_length);
/* destroys a plan made by jp_sino_plan_create or jp_lm_plan_create (jp_lm_plan_destroy is the same call) */
int jp_plan_destroy(jp_plan *plan);
/* jp_fwd / jp_back on the plan's LORs.  On a regular plan the track tiles are dealt per track
 * (tracks of any length, e.g. 36 rings: 1296 = 768 + 528 LORs) and read 16 bytes per track and the axial pattern
 * instead of 24 bytes per LOR.  (The unplanned jp_fwd / jp_back find tracks only where 768 consecutive LORs of the
 * list share their transaxial end points; they keep no state between calls.) */
int jp_fwd_planned(const jp_plan *plan, const float *img, const jp_geom *geom, float *p, void *stream);
int jp_back_planned(const jp_plan *plan, const float *y, const jp_geom *geom, float *img, void *stream);
/* jp_fwd_tof_sino / jp_back_tof_sino on the plan's LORs.  On a regular plan: track tiles --
 * the image rows of a track are interpolated along q1 once per tile in shared memory, the adjoint is staged in
 * shared memory (fixed point; a tile whose y holds Inf / NaN takes the per-LOR float path, so non-finite values
 * propagate as in the unplanned call) and flushed with 128-bit atomic adds. */
int jp_fwd_tof_sino_planned(const jp_plan *plan, const float *img, const jp_geom *geom, const jp_tof *tof, float *p,
                            void *stream);
int jp_back_tof_sino_planned(const jp_plan *plan, const float *y, const jp_geom *geom, const jp_tof *tof, float *img,
                             void *stream);
/* jp_sino_sens_tof / jp_sino_osem_tof on the plan's LORs (same arguments otherwise; workspace as for the unplanned
 * calls, only touched when the plan is not regular, a subset boundary cuts a track, or the TOF kernel is too wide) */
int jp_sino_sens_tof_planned(const jp_plan *plan, const int64_t *subset_offsets, int n_subsets, const float *mult,
                             const jp_geom *geom, const jp_tof *tof, float *sens, void *workspace, size_t workspace_bytes,
                             void *stream);
int jp_sino_osem_tof_planned(const jp_plan *plan, const int64_t *subset_offsets, int n_subsets, const float *y,
                             const float *mult, const float *contam, const float *sens, const jp_geom *geom,
                             const jp_tof *tof, float *img, int n_iter, void *workspace, size_t workspace_bytes, void *stream);

/* ---- hybrid mode: HOST pointers in and out, over all visible GPUs --------------------------- */
/* "data transfer from the host to all available GPUs, execution of projection kernels on the GPUs, and transfer of
 * the results back".  A jp_hybrid handle owns one worker per device it was created over (a host thread
 * per call, a CUDA stream, device buffers that are KEPT between calls and freed with the handle).
 *   devices   ordinals of the devices to use, n_devices of them; NULL = all visible devices.  A device may be listed
 *             more than once (several workers on one GPU).
 *   jp_hybrid_set_lors  splits the HOST LOR list into one contiguous shard per worker (cut at multiples of the list's
 *             track length when it has one, and of 768 LORs), uploads every shard ONCE and builds the shard's plan: a
 *             sinogram plan, or, when tofbin_host is given, a listmode plan (then geom and tof are required; they are
 *             the geometry / TOF model of the later jp_hybrid_*_tof_lm calls).  The host arrays are not kept.
 *   projection calls    move only what changes: the image to every GPU, the per-LOR values of each shard, the results
 *             back.  Forward results are disjoint; a back projection sums the workers' partial images on the host in
 *             worker order and ACCUMULATES the sum into img_host.  Same per-LOR arithmetic as the device calls.
 * All jp_hybrid_* calls return after their result is in host memory (they synchronise their own streams only), may
 * allocate device and pinned host memory, and do not change the calling thread's current device.  One call at a
 * time per handle.  Page-locked host arrays make the copies faster; pageable ones work. */
typedef struct jp_hybrid jp_hybrid;
int jp_hybrid_create(const int *devices, int n_devices, jp_hybrid **handle);
int jp_hybrid_destroy(jp_hybrid *handle);
int jp_hybrid_worker_count(const jp_hybrid *handle); /* -1 for NULL */
int jp_hybrid_set_lors(jp_hybrid *handle, const jp_lors *lors_host, const int16_t *tofbin_host /* or NULL */,
                       const jp_geom *geom /* with tofbin_host */, const jp_tof *tof /* with tofbin_host */);
int jp_hybrid_fwd(jp_hybrid *handle, const float *img_host, const jp_geom *geom, float *p_host);
int jp_hybrid_back(jp_hybrid *handle, const float *y_host, const jp_geom *geom, float *img_host);
int jp_hybrid_fwd_tof_sino(jp_hybrid *handle, const float *img_host, const jp_geom *geom, const jp_tof *tof, float *p_host);
int jp_hybrid_back_tof_sino(jp_hybrid *handle, const float *y_host, const jp_geom *geom, const jp_tof *tof, float *img_host);
int jp_hybrid_fwd_tof_lm(jp_hybrid *handle, const float *img_host, float *p_host);
int jp_hybrid_back_tof_lm(jp_hybrid *handle, const float *y_host, float *img_host);

/* One-shot forms (same semantics as jp_fwd / jp_back / ..., every pointer -- inside lors_host too -- a HOST pointer):
 * each makes a handle over all visible devices, sets the list, projects and destroys the handle.  jp_back*_host
 * ACCUMULATE into img_host.  Callers that project a list more than once should keep a handle instead. */
int jp_fwd_host(const jp_lors *lors_host, const float *img_host, const jp_geom *geom, float *p_host);
int jp_back_host(const jp_lors *lors_host, const float *y_host, const jp_geom *geom, float *img_host);
int jp_fwd_tof_sino_host(const jp_lors *lors_host, const float *img_host, const jp_geom *geom, const jp_tof *tof,
                         float *p_host);
int jp_back_tof_sino_host(const jp_lors *lors_host, const float *y_host, const jp_geom *geom, const jp_tof *tof,
                          float *img_host);
int jp_fwd_tof_lm_host(const jp_lors *lors_host, const int16_t *tofbin_host, const float *img_host, const jp_geom *geom,
                       const jp_tof *tof, float *p_host);
int jp_back_tof_lm_host(const jp_lors *lors_host, const int16_t *tofbin_host, const float *y_host, const jp_geom *geom,
                        const jp_tof *tof, float *img_host);

/* ---- misc ----------------------------------------------------------------------------------------- */
/* text of the last CUDA error seen by the calling thread ("" if none); valid until the next call */
const char *jp_last_error(void);
/* library version, e.g. 100 = 0.1.0 */
int jp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* JOSEPH_B200_H */
