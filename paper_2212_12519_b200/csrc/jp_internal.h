// jp_internal.h -- launcher declarations shared by the translation units of libjoseph_b200.so
#pragma once
#include <cstddef>
#include <cstdint>
#include <cuda_runtime.h>

#include "jp_ray.cuh"

namespace jp {

// LOR index of work item c is j = first + c * stride (c = 0..count-1); per-LOR inputs/outputs
// (p, y, tofbin) are indexed by j when `compact` is false and by c when it is true.
// per-thread error text returned by jp_last_error() (512 bytes)
char *err_buf();

struct Range {
    int64_t first, stride, count;
    bool compact;
    const int *perm = nullptr; // if set (and not compact): per-LOR inputs/outputs are indexed by perm[j]
    int64_t io_off = 0;        // compact: per-LOR inputs/outputs are indexed by c + io_off
};

cudaError_t launch_classify(const Lors &l, int64_t n, uint8_t *axis, cudaStream_t st);

cudaError_t launch_plane_steps(const Lors &l, int64_t n, const Geom &g, unsigned long long *total, cudaStream_t st);

cudaError_t launch_plane_steps_tof_lm(const Lors &l, const int16_t *tofbin, int64_t n, const Geom &g, const Tof &t,
                                      unsigned long long *total, cudaStream_t st);

cudaError_t launch_fwd(const Lors &l, Range rg, const float *img, const Geom &g, float *p, cudaStream_t st);
cudaError_t launch_back(const Lors &l, Range rg, const float *y, const Geom &g, float *img, cudaStream_t st);

// tiled non-TOF kernels (jp_tile.cu): track tiles through shared memory, everything else per LOR
// pv: a REGULAR sinogram plan (tiles per track, `l` is not read), or null: tiles of 768 consecutive LORs of `l`
struct SinoPlanView;
cudaError_t launch_fwd_tile(const Lors &l, int64_t n, const float *img, const Geom &g, float *p, cudaStream_t st,
                            const SinoPlanView *pv = nullptr, int lane_map = 1);
cudaError_t launch_back_tile(const Lors &l, int64_t n, const float *y, const Geom &g, float *img, cudaStream_t st,
                             const SinoPlanView *pv = nullptr, int lane_map = 1);

// table of the TOF edge function (jp_tof_lut.cu): stream-ordered device scratch, one per call
cudaError_t tof_lut_create(const Tof &t, cudaStream_t st, TofLut *out);
void tof_lut_destroy(TofLut *lut, cudaStream_t st);

cudaError_t launch_fwd_tof_sino(const Lors &l, Range rg, const float *img, const Geom &g, const Tof &t,
                                const TofLut &lut, float *p, cudaStream_t st);
cudaError_t launch_back_tof_sino(const Lors &l, Range rg, const float *y, const Geom &g, const Tof &t,
                                 const TofLut &lut, float *img, cudaStream_t st);

// sliding-window TOF sinogram kernels (jp_tof_sino.cu); cudaErrorNotSupported: window wider than compiled
// optional fused stages of the sliding-window kernels (all pointers may be null = plain projection):
//   forward, y_em set: the OSEM ratio  r = mult y_em / (mult p + contam) if that > 1e-9 else 0  is written
//                      instead of p (reading S2; mult per LOR, contam per LOR and bin, either may be null);
//   back, mult_bcast set: the value of every bin of LOR j is mult_bcast[j] (sensitivity image A^T (mult x 1)),
//                      y is not read.
struct SinoEpi {
    const float *y_em = nullptr;
    const float *mult = nullptr;
    const float *contam = nullptr;
    const float *mult_bcast = nullptr;
    int ones_bcast = 0; // back: every bin of every LOR is 1 (sensitivity without multiplicative factors)
};

cudaError_t launch_tof_sino_win(bool back, const Lors &l, int64_t n, const float *pimg_r, float *pimg_w, const Geom &g,
                                const Tof &t, float *p, const float *y, cudaStream_t st, const SinoEpi *epi = nullptr);

// one OSEM subset pass in one kernel: pimg_w += A^T (mult y / (mult A pimg_r + contam)); epi.y_em must be set
cudaError_t launch_tof_sino_osem(const Lors &l, int64_t n, const float *pimg_r, float *pimg_w, const Geom &g, const Tof &t,
                                 const SinoEpi &epi, cudaStream_t st);

// r <- mult y / (mult r + contam) (reading S2) and r <- mult broadcast over the bins: the unfused stages used
// with the generic TOF sinogram kernels
cudaError_t launch_sino_ratio(float *r, const float *y, const float *mult, const float *contam, int64_t n, int nbins,
                              cudaStream_t st);
cudaError_t launch_sino_bcast(float *r, const float *mult, int64_t n, int nbins, cudaStream_t st);

// lm_mode: 0 = p = A x;  1 = p = (A x > 1e-9) ? 1/(A x) : 0   (OSEM ratio fused into the epilogue)
cudaError_t launch_fwd_tof_lm(const Lors &l, const int16_t *tofbin, Range rg, const float *img, const Geom &g,
                              const Tof &t, const TofLut &lut, float *p, int lm_mode, cudaStream_t st);
cudaError_t launch_back_tof_lm(const Lors &l, const int16_t *tofbin, Range rg, const float *y, const Geom &g,
                               const Tof &t, const TofLut &lut, float *img, cudaStream_t st);

// zero-padded image copies for the per-LOR kernels (jp_pad.cu)
int64_t padded_voxels(const Geom &g);
cudaError_t padded_create(const float *img, const Geom &g, bool zero_only, cudaStream_t st, float **out);
cudaError_t padded_add_to(const float *pimg, const Geom &g, float *img, cudaStream_t st);
void padded_destroy(float *p, cudaStream_t st);
cudaError_t launch_osem_update_padded(float *x, float *px, float *pb, const float *sens, float scale, const Geom &g,
                                      cudaStream_t st);

// quad image / accumulators and the TOF listmode kernels on them (jp_quad.cu); q0: q1 = axis 1 (principal
// axis 0), q1: q1 = axis 0 (principal axis 1); each array has padded_voxels(g) float4 elements
cudaError_t launch_quad_build(const float *img, const Geom &g, float4 *q0, float4 *q1, cudaStream_t st);
cudaError_t launch_quad_merge(const float4 *b0, const float4 *b1, const Geom &g, float *img, cudaStream_t st);
cudaError_t launch_quad_osem_update(float *x, const float4 *b0, const float4 *b1, float *extra, const float *sens,
                                    float scale, const Geom &g, cudaStream_t st);
cudaError_t launch_fwd_tof_lm_quad(const Lors &l, const int16_t *tofbin, Range rg, const float4 *q, const Geom &g,
                                   const Tof &t, const TofLut &lut, float *p, int lm_mode, cudaStream_t st);
// forward + ratio + back of one OSEM subset in one pass (quad image in, quad accumulator out)
cudaError_t launch_osem_tof_lm_quad(const Lors &l, const int16_t *tofbin, Range rg, const float4 *q, const Geom &g,
                                    const Tof &t, const TofLut &lut, float4 *b, cudaStream_t st);
// y_mode 1: y holds the forward sums without the factor cf; the OSEM ratio 1 / (cf y) is back projected
// gt: TOF weights from this G1 table (jp_g1tab.cuh: the table of the brick / line-tile kernels) instead of `lut`
struct G1Tab;
cudaError_t launch_back_tof_lm_quad(const Lors &l, const int16_t *tofbin, Range rg, const float *y, const Geom &g,
                                    const Tof &t, const TofLut &lut, float4 *b, cudaStream_t st, int y_mode = 0,
                                    const G1Tab *gt = nullptr);

// TOF listmode on line tiles (jp_lm_tile.cu): events [first, first + count) of a SORTED list; outputs / inputs at
// perm[e] (perm != null) or io_off + e - first; cudaErrorNotSupported: image too wide for the tiled kernels
cudaError_t launch_fwd_tof_lm_tile(const Lors &l, const int16_t *tofbin, int64_t first, int64_t count, const int *perm,
                                   int64_t io_off, const float *img, const Geom &g, const Tof &t, float *p, int lm_mode,
                                   cudaStream_t st);

cudaError_t launch_back_tof_lm_tile(const Lors &l, const int16_t *tofbin, int64_t first, int64_t count, const int *perm,
                                    int64_t io_off, const float *y, const Geom &g, const Tof &t, float *img,
                                    cudaStream_t st);

bool lm_tile_supported(const Geom &g, const Tof &t, bool tof);

// listmode plan (jp_plan.cu)
struct LmPlan;
cudaError_t lm_plan_create(const Lors &l, const int16_t *tofbin, int64_t n, const Geom &g, const Tof &t,
                           int n_subsets, cudaStream_t st, LmPlan **out);
void lm_plan_destroy(LmPlan *pl);
int64_t lm_plan_n(const LmPlan *pl);
int64_t lm_plan_runs(const LmPlan *pl); // runs of sorted events sharing their transaxial line
int lm_plan_subsets(const LmPlan *pl);
int lm_plan_path(const LmPlan *pl);            // 0: chosen from the run statistics, 1: line tiles, 2: quad image
void lm_plan_set_path(LmPlan *pl, int path);
const Geom &lm_plan_geom(const LmPlan *pl);
const Tof &lm_plan_tof(const LmPlan *pl);
void lm_plan_view(const LmPlan *pl, int m, bool compact, Lors *l, const int16_t **tb, Range *rg);
// events of subset m with principal axis a (a contiguous run of the sorted list): first index and count
void lm_plan_segment(const LmPlan *pl, int m, int a, int64_t *first, int64_t *count);
// the planned TOF listmode projectors (jp_api.cu), subset < 0: all events; p / y in caller order
// sorted_io: p / y are in PLAN order (index = position in the sorted list) instead of caller order
cudaError_t lm_plan_fwd_tof(LmPlan *pl, int subset, const float *img, float *p, cudaStream_t st, bool sorted_io = false);
cudaError_t lm_plan_back_tof(LmPlan *pl, int subset, const float *y, float *img, cudaStream_t st, bool sorted_io = false);
// out[k] = in[perm[k]] (to plan order) or out[perm[k]] = in[k] (to caller order)
cudaError_t lm_plan_permute(const LmPlan *pl, const float *in, float *out, bool to_plan_order, cudaStream_t st);
// persistent quad scratch of the plan (allocated on first use): which = 0,1: Q0,Q1; 2,3: B0,B1
cudaError_t lm_plan_quad(LmPlan *pl, int which, float4 **out);

// listmode bricks (jp_brick.cu): the events of every subset cut into pieces per image brick, see the file header
struct BrickSet;
bool brick_supported(const Geom &g, const Tof &t, int n_subsets);
cudaError_t brick_set_create(const Lors &l, const int16_t *tb, int64_t n, const Geom &g, const Tof &t, int n_subsets,
                             const int64_t *sub_first, const int64_t *sub_count, cudaStream_t st, BrickSet **out);
void brick_set_destroy(BrickSet *bs);
int64_t brick_set_pieces(const BrickSet *bs);
float *brick_set_acc(const BrickSet *bs); // one float per event: scratch of the planned forward projection
cudaError_t lm_plan_bricks(LmPlan *pl, cudaStream_t st, const BrickSet **out);
// acc[e - ev0] += sum_k G(k) bilinear(k) over the pieces of subset m (ev0: sorted position of the subset's first event)
// table: the G1 table of t if the caller already has one (else made and freed here, stream-ordered)
cudaError_t launch_brick_fwd(const BrickSet *bs, int m, const float *img, const Geom &g, const Tof &t, int64_t ev0, float *acc,
                             cudaStream_t st, const G1Tab *table = nullptr);
// p[perm ? perm[e] : e - first + io_off] = cf acc[e - ev0] (mode 0) or its OSEM ratio (mode 1), e in [first, first + count)
cudaError_t launch_brick_finish(const BrickSet *bs, const float *acc, int64_t first, int64_t count, int64_t ev0, const int *perm,
                                int64_t io_off, int mode, float *p, cudaStream_t st);

// sinogram plan (jp_sino_plan.cu): a LOR list analysed once.  REGULAR = K tracks of T LORs each (a track: identical
// transaxial end points) that all share ONE axial pattern (zs, ze)[T] -- every sinogram of a ring scanner.  A regular
// plan keeps only the K transaxial end-point quadruples, the pattern and a lane order (pattern indices sorted by
// |ze - zs|: LORs of equal axial tilt have identical TOF weights on every plane); any other list is kept as a copy.
constexpr int kSinoSlice = 384;    // LORs of a track one CTA of the tile kernels takes (jp_tof_sino_tile.cu)
constexpr int kSinoGroupsMax = 16; // groups of equal |ze - zs| per slice that get shared TOF weight rows
struct SinoPlan;
struct SinoPlanView {
    int64_t n = 0;        // LORs
    int64_t K = 0;        // tracks (regular)
    int T = 0;            // LORs per track (regular)
    int regular = 0;
    double dz_max = 0.0;  // max |ze - zs| of the pattern
    const float4 *trk = nullptr;  // [K] (xs, ys, xe, ye)
    const float2 *zpat = nullptr; // [T] (zs, ze)
    // lane order: the pattern indices arranged in slices of kSinoSlice entries; a slice is made of whole GROUPS (LORs
    // of equal |ze - zs|, ordered by sign and zs) wherever they fit, at most kSinoGroupsMax of them
    const int *order = nullptr;            // [T]
    const unsigned char *slot_grp = nullptr; // [T] group of the entry, numbered from 0 inside its slice
    const int *slice_ng = nullptr;         // [ceil(T / kSinoSlice)] groups of the slice; 0: too many, weights per lane
    int slice_len = kSinoSlice;
    // whole-track kernels (jp_track.cu): a track is cut into t_npieces equal pieces of at most 2304 LORs, a piece has
    // t_npt x 256 slots; [0] forward lane order, [1] adjoint lane order
    const float2 *t_zp[2] = {nullptr, nullptr}; // [t_npieces][slots] (zs, ze) of the slot's LOR
    const int *t_ord[2] = {nullptr, nullptr};   // [t_npieces][slots] its index inside the track, -1: empty slot
    int t_npieces = 0, t_npt = 0;
    Lors lors{};                  // irregular: the plan's own SoA copy of the list
};
cudaError_t sino_plan_create(const Lors &l, int64_t n, cudaStream_t st, SinoPlan **out);
void sino_plan_destroy(SinoPlan *pl);
SinoPlanView sino_plan_view(const SinoPlan *pl);
// regular plan: write the end points of LORs [first, first + count) as SoA arrays into coord6 (6 x count floats)
cudaError_t sino_plan_expand(const SinoPlanView &pv, int64_t first, int64_t count, float *coord6, cudaStream_t st, Lors *out);

// non-TOF projections of a REGULAR plan, one CTA per track (jp_track.cu); cudaErrorNotSupported: image too wide
cudaError_t launch_fwd_track(const SinoPlanView &pv, const float *img, const Geom &g, float *p, cudaStream_t st);
cudaError_t launch_back_track(const SinoPlanView &pv, const float *y, const Geom &g, float *img, cudaStream_t st);

// TOF sinogram kernels on the track tiles of a REGULAR plan (jp_tof_sino_tile.cu), tracks [k0, k0 + nk):
//   mode 0  p[j][:] = A x            (p, y, epi arrays are indexed by the LOR index j of the plan's list)
//   mode 1  img_w += A^T y           (or the broadcast values of epi: sensitivity images)
//   mode 2  img_w += A^T (mult y_em / (mult A img_r + contam))   one OSEM subset pass (epi.y_em set)
// img_r / img_w: UNPADDED images.  cudaErrorNotSupported: TOF window wider than compiled, or image too wide.
cudaError_t launch_tof_sino_tile(int mode, const SinoPlanView &pv, int64_t k0, int64_t nk, const float *img_r, float *img_w,
                                 const Geom &g, const Tof &t, float *p, const float *y, const SinoEpi *epi, cudaStream_t st);

// window bins the TOF sinogram kernels are compiled for (0: TOF kernel too wide); R = n_sigmas sigma / W + 1/2
int tof_window_bins(const Tof &t, double *R_out);

// resolution model (jp_gauss.cu): out = G in, three separable passes; tmp = nvox floats of scratch; in may alias out
cudaError_t launch_gauss3d(const float *in, float *out, float *tmp, const Geom &g, float sigma_mm, float nsig,
                           cudaStream_t st);
cudaError_t launch_add_clear(float *a, float *b, int64_t n, cudaStream_t st); // a += b; b = 0

// x = sens > 0 ? x * b * scale / sens : 0;  b = 0   (OSEM multiplicative update, clears b for the next subset)
cudaError_t launch_osem_update(float *x, float *b, const float *sens, float scale, int64_t nvox, cudaStream_t st);

} // namespace jp
