// Internal declarations of libcbct (CUDA path).  Not part of the ABI; see include/cbct.h.
#pragma once
#include <cuda_runtime.h>

#include <atomic>
#include <functional>

#include <cstdint>
#include <cmath>
#include <cstdio>
#include <algorithm>
#include <vector>

#include "../../include/cbct.h"

// ------------------------------------------------------------------------------------------
// Device-side geometry.  Every ray is traversed slab by slab along its MAJOR axis: x if
// |dX| >= |dY| in voxel units (class 0), else y (class 1); the other in-plane axis is MINOR.
// |d minor / d major| <= 1 by construction, so a ray crosses at most one minor plane per slab.
// ------------------------------------------------------------------------------------------
constexpr int kPadLo = 4;      // zero floats before minor index 0 in the padded copies (>= 2; 4 keeps rows 16-B aligned)
constexpr int kPadHi = 2;      // zero floats after minor index nmin-1 (>= 2)
constexpr int kPadK = 2;       // zero planes below k = 0 and above k = nz-1

// Per-(angle,u) constants, computed in fp64 on the host.  32 bytes = two 16-byte loads.
struct __align__(16) RayXY {
    float mc;       // minor coordinate (voxel units, minus joff) where the ray meets major plane ioff
    float sm;       // d(minor)/d(major), voxel units
    float inv_sm;   // 1/sm (+1e30 if sm == 0)
    float tc;       // ray parameter t in [0,1] at major plane ioff
    float dt;       // dt per major voxel (signed)
    float inv_dt;   // 1/dt
    float lxy2;     // hmaj^2 + (sm hmin)^2  [mm^2]; chord per slab = sqrt(lxy2 + (dt Dz)^2)
    int range;      // bits 0-14 ilo, 15-29 ihi (slabs where the ray can touch minor range [-1,nmin+1]), bit 30 class
};
__host__ __device__ inline int ray_ilo(int r) { return r & 0x7fff; }
__host__ __device__ inline int ray_ihi(int r) { return (r >> 15) & 0x7fff; }
__host__ __device__ inline int ray_cls(int r) { return (r >> 30) & 1; }

// Per-class view of the volume grid (class 0: major x / minor y; class 1: major y / minor x).
struct ClassGrid {
    int nmaj, nmin, ioff, joff;
    float hmaj, hmin;
    int row_stride;             // floats per padded minor row
    long long plane_stride;     // floats per padded k-plane = nmaj * row_stride
};

struct DevGeom {
    int na, nu, nv, nx, ny, nz;
    int koff;                   // nz / 2
    float zfrac;                // nz/2.0 - koff  (0 or 0.5)
    float hx, hy, hz, du, dv, sad, sdd;
    float cu, cv;               // detector index of the central ray: (nu-1)/2 - off_u/du, (nv-1)/2 - off_v/dv
    float cv_lo;                // the part of that v index the float cv drops (0 for a centred panel)
    float hzdv_hi, hzdv_lo;     // hz / dv as an unevaluated sum of two floats (the gather places z planes on the detector with it)
    ClassGrid cls[2];
    const RayXY *rays;          // [na][nu]
    const float4 *rays_lo;      // [na][nu]  what the floats mc, sm, tc of RayXY drop of their fp64 values (x, y, z); read by the gather
    const float *zeta;          // [nv]  Dz(v)/hz
    const float *inv_zeta;      // [nv]  hz/Dz(v) (+-1e30 if Dz == 0)
    const float *dz_mm;         // [nv]  Dz(v) in mm
    const float2 *cs;           // [na]  (cos, sin)
};

// Host-side handle.
struct cbct_geometry {
    // user geometry (fp64)
    double sad, sdd, du, dv, hx, hy, hz;
    double off_u = 0.0, off_v = 0.0;          // in-plane shift of the detector panel, mm (NEXT-3, Q19)
    int na, nu, nv, nx, ny, nz;
    std::vector<double> angles;

    DevGeom dev{};
    // device tables
    RayXY *d_rays = nullptr;
    float4 *d_rays_lo = nullptr;
    float *d_zeta = nullptr, *d_inv_zeta = nullptr, *d_dz = nullptr;
    float2 *d_cs = nullptr;
    int2 *d_tiles[2] = {nullptr, nullptr};   // forward work list per class: (angle, u0)
    int n_tiles[2] = {0, 0};
    int n_tiles_half[2] = {0, 0};             // tiles of the first half turn (angle index < na/2): the twin march launches only these
    int last_march_twin = 0;                  // the last projection on this handle was made by the twin march (op_residual follows it)
    bool twin_ok = false;                     // angle a + na/2 = angle a + 180 degrees for every a < na/2 (and mirror symmetry switched on)
    unsigned char *d_angle_has[2] = {nullptr, nullptr};   // [na] does this angle have rays of the class
    std::vector<unsigned char> h_angle_has[2];
    float max_abs_sz = 0.f;
    float bp_run_max = 2.f;                   // upper bound of the detector rows one voxel row's run can hold (fixed-point prefix sums)

    // lazily allocated scratch (device)
    float *vol_pad[2] = {nullptr, nullptr};   // padded [nz+2K][nmaj][row_stride] copies (class 0 transposed)
    float *proj_tmp = nullptr;                // scaled residual / projections
    float2 *proj_prefix = nullptr;            // [na][nv+1][nu] compensated prefix sums of proj_tmp along v
    float *G_cls[2] = {nullptr, nullptr};     // per-class backprojection outputs (class 0 in [k][i][j] order)
    float *vol_a = nullptr, *vol_b = nullptr, *vol_c = nullptr, *vol_f = nullptr;   // g, u ping-pong, f
    float *Y_level = nullptr;                 // binned data for a coarse level
    float *vc_tau = nullptr, *vc_f0 = nullptr, *vc_d = nullptr, *vc_e = nullptr;   // V-cycle: tau, restricted iterate, gradient, scratch
    float *fdk_q = nullptr;                   // FDK: pre-weighted, filtered projections
    double *fdk_hk = nullptr;                 // FDK: ramp taps D h[k], k odd
    double2 *fdk_cs = nullptr;                // FDK: (cos, sin) of the views in fp64
    double *red_partial = nullptr;            // reduction partials
    double *red_out = nullptr;                // 2 doubles
    double *h_red = nullptr;                  // pinned host mirror of red_out
    float *host_stage_vol = nullptr, *host_stage_proj = nullptr, *host_stage_vol2 = nullptr;  // device staging for *_host
    unsigned long long bytes = 0;
    struct Guarded { void *ptr; size_t bytes, padded; };
    std::vector<Guarded> guarded;             // buffers allocated in guard mode (cbct_set_guard_mode): user pointer, sizes

    // TV sweep (tv_tma.cu): encoded tensor maps of the volumes the sweeps read, keyed by (pointer, box); the dims are the
    // handle's.  A map depends on nothing else, so an entry stays valid even if the caller frees and reuses the address.
    struct TmapSlot { const void *ptr = nullptr; unsigned bx = 0, by = 0; alignas(64) unsigned char map[128]; };
    TmapSlot tv_tmaps[8];
    int tv_tmap_next = 0;                     // round-robin replacement

    int bp_parts = 1, G_parts_alloc[2] = {0, 0};   // gather: angle parts per column chunk (small volumes), partial volumes allocated
    int bp_mode = 0;                          // step 1 of A1: 0 exact transpose, 1 eq. 2 (cbct_set_backprojector)
    int use_mirror = 1;                        // march and gather: use the scan's mirror symmetry about z = 0 where it has one (cbct_set_mirror_symmetry)
    int fw_staged = 0;                        // projector: 1 = TMA-staged bricks (projector_tma.cu), 0 = __ldg march
    int fw_bj[2] = {0, 0}, fw_bk[2] = {0, 0};  // brick spans per class (0 = not computed yet)
    int bin_detector = 1;                     // coarse levels bin the detector 2x2 (O6) or keep it at full resolution (Q20)

    cudaStream_t copy_stream = nullptr;       // host-buffer path: the upload of Y runs here, beside the first kernels (api.cu)
    cudaEvent_t ev_f0 = nullptr, ev_Y = nullptr;
    cudaStream_t graph_stream = nullptr;      // internal stream the outer iteration of a small volume is captured on (api.cu)
    unsigned long long launches_per_iteration = 0;   // kernels one outer iteration launches (counted on an eager one)

    // multigrid
    cbct_geometry *coarse = nullptr;
    int coarsen_flags[4] = {0, 0, 0, 0};
    bool coarse_tried = false;

    size_t n_vox() const { return (size_t)nx * ny * nz; }
    size_t n_proj() const { return (size_t)na * nu * nv; }
};

// ---- error handling -----------------------------------------------------------------------
void cbct_set_error(const char *fmt, ...);
#define CBCT_CUDA(call)                                                                         \
    do {                                                                                        \
        cudaError_t e_ = (call);                                                                \
        if (e_ != cudaSuccess) {                                                                \
            cbct_set_error("%s:%d: %s -> %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
            return CBCT_ERR_CUDA;                                                               \
        }                                                                                       \
    } while (0)
#define CBCT_TRY(call)                        \
    do {                                      \
        cbct_status s_ = (call);              \
        if (s_ != CBCT_OK) return s_;         \
    } while (0)

extern std::atomic<unsigned long long> g_cbct_launches;
#define CBCT_LAUNCH_CHECK()                                                      \
    do {                                                                         \
        ++g_cbct_launches;                                                       \
        cudaError_t e_ = cudaGetLastError();                                     \
        if (e_ != cudaSuccess) {                                                 \
            cbct_set_error("%s:%d: kernel launch -> %s", __FILE__, __LINE__, cudaGetErrorString(e_)); \
            return CBCT_ERR_CUDA;                                                \
        }                                                                        \
    } while (0)

// ---- per-kernel-class event timing (profile.cu) ---------------------------------------------
bool cbct_profile_is_on();
struct ProfileScope {
    ProfileScope(int tag, cudaStream_t st);
    ~ProfileScope();
    int tag_;
    cudaStream_t st_;
    cudaEvent_t a_;
};

// ---- scratch ------------------------------------------------------------------------------
// zero = true clears the new buffer with cudaMemsetAsync on `st`, the stream of the first kernel that will use it
cbct_status cbct_dev_alloc(cbct_geometry *g, void **p, size_t bytes, bool zero, cudaStream_t st);
void cbct_dev_free(cbct_geometry *g, void *p);
template <typename T>
inline cbct_status ensure(cbct_geometry *g, T **p, size_t count)
{
    if (*p) return CBCT_OK;
    return cbct_dev_alloc(g, (void **)p, count * sizeof(T), false, nullptr);
}
template <typename T>
inline cbct_status ensure_zeroed(cbct_geometry *g, T **p, size_t count, cudaStream_t st)
{
    if (*p) return CBCT_OK;
    return cbct_dev_alloc(g, (void **)p, count * sizeof(T), true, st);
}
inline size_t pad_elems(const cbct_geometry *g, int c)
{
    return (size_t)(g->nz + 2 * kPadK) * (size_t)g->dev.cls[c].plane_stride;
}

// ---- operators (device pointers, async on stream) ---------------------------------------------
// projector.cu
cbct_status op_pad_copies(cbct_geometry *g, const float *d_vol, cudaStream_t st);
// mode 0: out = P f ; mode 1: out = l * (P f - Y)  (scaled residual for the gather) ; mode 2: out = P f - Y
cbct_status op_forward_padded(cbct_geometry *g, float *d_out, const float *d_Y, int mode, cudaStream_t st);
// q (= P f from mode 0) -> l (q - Y) (mode 1) or q - Y (mode 2), in place: a2 on its own, bit-identical to the fused store
cbct_status op_residual(cbct_geometry *g, float *d_q, const float *d_Y, int mode, cudaStream_t st);
cbct_status op_forward_padded_tma(cbct_geometry *g, float *d_out, const float *d_Y, int mode, cudaStream_t st, int *done);   // projector_tma.cu
// backprojector.cu : gathers of the (already l-scaled) projections into G_cls[0], G_cls[1].
// op_backproject_prefix builds the prefix sums along v that the gather reads (scale != 0: of l * d_in,
// also written to d_rs_out); it must run on the same projections before op_backproject_gather.
cbct_status op_backproject_prefix(cbct_geometry *g, const float *d_in, int scale, float *d_rs_out, cudaStream_t st);
cbct_status op_backproject_gather(cbct_geometry *g, const float *d_scaled, cudaStream_t st);
// out = G1 + G0^T                         (f == nullptr)
// out = f - c (G1 + G0^T), optionally clamped at 0   (f != nullptr)
cbct_status op_combine(cbct_geometry *g, const float *f, float c, int clamp, float *out, cudaStream_t st);
// backprojector_eq2.cu : out = B r (eq. 2, f == nullptr) or out = f - c (B r) [clamped]
cbct_status op_backproject_eq2(cbct_geometry *g, const float *d_proj, const float *f, float c, int clamp, float *out,
                               cudaStream_t st);
// tv.cu
cbct_status op_tv_sweep(cbct_geometry *g, const float *u_in, const float *gv, float *u_out,
                        float beta, float eps, float dt, int clamp, cudaStream_t st);
cbct_status op_tv_sweep_rows(cbct_geometry *g, const float *u_in, const float *gv, float *u_out, float beta, float eps,
                             float dt, int clamp, cudaStream_t st, int *done);   // tv_rows.cu
cbct_status op_tv_sweep_tma(cbct_geometry *g, const float *u_in, const float *gv, float *u_out, float beta, float eps,
                            float dt, int clamp, cudaStream_t st, int *done);    // tv_tma.cu
cbct_status op_tv_value(cbct_geometry *g, const float *f, float eps, double *d_out, cudaStream_t st);
// transfers.cu
cbct_status op_prolong(cbct_geometry *fine, const float *c, float *f, cudaStream_t st);
cbct_status op_restrict(cbct_geometry *fine, const float *f, float *c, cudaStream_t st);
cbct_status op_bin2x2(cbct_geometry *fine, const float *y, float *yc, cudaStream_t st);
cbct_status op_sumsq_diff(cbct_geometry *g, const float *a, const float *b, size_t n, double *d_out, cudaStream_t st);
cbct_status op_tv_grad(cbct_geometry *g, const float *f, float eps, float *out, cudaStream_t st);   // tv.cu: out = grad TV_eps(f)
// api.cu: one level of A1 (tau: optional FAS term), the data gradient P^T (P f - Y) (or eq. 2's), E_eps (synchronises)
cbct_status op_fbs_level(cbct_geometry *g, const float *d_Y, float *f, int n_outer, int n_inner, float step, float mu, float eps,
                         float omega, double *trace, float rel_tol, int *iters, const float *tau, cudaStream_t st,
                         const std::function<cbct_status()> *y_gate = nullptr);   // y_gate: see api.cu (host-buffer path)
cbct_status op_data_gradient(cbct_geometry *g, const float *d_f, const float *d_Y, float *d_G, cudaStream_t st);
cbct_status op_energy(cbct_geometry *g, const float *d_f, const float *d_Y, float mu, float eps, double *out3, cudaStream_t st);
cbct_status op_axpy_clamp(cbct_geometry *g, const float *f, const float *G, float c, int clamp, float *out, cudaStream_t st);
