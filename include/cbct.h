/*
 * cbct.h — C ABI of libcbct.so: the B200-native (sm_100a) hot path of TV-regularised cone-beam
 * CT reconstruction by forward-backward splitting (Jia, Lou, Li, Song, Jiang, arXiv 1002.3675).
 *
 * Citations: P:<n> = PAPER.md line n (the paper); O<n>/Q<n> = the readings in DESIGN.md
 * (the paper leaves the discretisation open; every choice is listed there).
 *
 * Conventions (all entry points)
 *   - Lengths in mm, angles in radians.  Rotation axis z.  Source S(t) = (SAD cos t, SAD sin t, 0);
 *     detector centre -(SDD-SAD)(cos t, sin t, 0); detector axes u^ = (-sin t, cos t, 0), v^ = z^;
 *     pixel (iu,iv) centre at ((iu-(nu-1)/2) du, (iv-(nv-1)/2) dv); volume centred at the origin.
 *   - Volume layout   f[k][j][i]  (x fastest), nz*ny*nx floats.
 *     Projection layout Y[a][iv][iu] (u fastest), n_angles*nv*nu floats.
 *   - Pointers named d_* are DEVICE pointers to contiguous fp32 memory owned by the caller
 *     (e.g. a PyTorch CUDA tensor); pointers named h_* are HOST pointers.  The library never frees
 *     or reallocates caller memory.  Inputs and outputs must not alias unless stated.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Device
 *     entry points are asynchronous on that stream; they synchronise with the host only where
 *     stated.  The *_host entry points copy host<->device on that stream and return after
 *     synchronising it.
 *   - A handle owns per-angle ray tables and lazily allocated scratch (grown on first use, freed
 *     by cbct_geometry_destroy).  A handle must not be used from two host threads or two streams
 *     at the same time.  One CUDA device per process (the intended deployment is one process per GPU): kernel
 *     attributes and occupancy figures are cached per process, the launch counter and the optional per-kernel timing
 *     (cbct_profile_*) are process-wide.
 *   - Errors: every call returns a cbct_status; nothing throws or aborts across the ABI.  On
 *     failure outputs are unspecified and cbct_last_error() describes the failure (thread-local).
 *   - There is no CPU fallback: with no CUDA device every compute call returns CBCT_ERR_CUDA.
 */
#ifndef CBCT_H
#define CBCT_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cbct_geometry cbct_geometry;   /* opaque, library-owned */

typedef enum {
    CBCT_OK = 0,
    CBCT_ERR_INVALID_ARG = 1,   /* NULL required pointer, non-positive size or parameter */
    CBCT_ERR_SHAPE = 2,         /* geometry the kernels do not support (see cbct_geometry_create), odd
                                   dimension on an axis that must coarsen */
    CBCT_ERR_ALLOC = 3,         /* host or device allocation failed */
    CBCT_ERR_CUDA = 4           /* a CUDA runtime call or kernel launch failed, or no device */
} cbct_status;

/*
 * Scan geometry ("an operator P^theta projects f onto an x-ray imager plane in a cone beam
 * geometry at an angle theta"; convention O0).
 *   sad_mm, sdd_mm     source-axis and source-detector distance (L0 of P:99); 0 < sad < sdd
 *   h_angles_rad       HOST array of n_angles projection angles, any list (360 deg equi-spaced P:119,
 *                      200 deg arc P:121); copied
 *   nu, nv, du, dv     detector pixels and pitch ("512 x 384 detectors" = nu x nv)
 *   nx..nz, hx..hz     volume dims and voxel size
 * Builds the per-(angle,u) ray tables (fp64 on the host, stored fp32 on the device).
 * Errors: INVALID_ARG for NULL / non-positive values or sad >= sdd; SHAPE if the volume's
 * circumscribed cylinder is not strictly between source and detector, if a dimension exceeds
 * 16384, if a padded volume copy ((nz+4) * nx * (ny+8) elements, or with x and y swapped) or
 * n_angles * (nv+1) * nu reaches 2^31 elements (32-bit offsets in the kernels), or if some ray climbs more than 0.999 voxels in z per voxel of its major (x or y) axis
 * (the slab march assumes at most one z-plane crossing per slab; true for every cone-beam CT
 * geometry with hz not much smaller than hx, hy).  No device memory is touched if this fails.
 */
cbct_status cbct_geometry_create(double sad_mm, double sdd_mm,
                                 const double *h_angles_rad, int n_angles,
                                 int nu, int nv, double du_mm, double dv_mm,
                                 int nx, int ny, int nz, double hx_mm, double hy_mm, double hz_mm,
                                 cbct_geometry **out);

/*
 * NEXT-3 (reading Q19): the same with the detector panel shifted in its own plane by (off_u_mm, off_v_mm): pixel (iu,iv)
 * sits at ((iu-(nu-1)/2) du + off_u, (iv-(nv-1)/2) dv + off_v) about the point where the central ray meets the imager
 * (half-fan scans shift the panel along u; the paper's scans are centred full-fan).  Source, central ray and L0 = sdd
 * are unchanged; coarse levels keep the shift.  Zero offsets give exactly cbct_geometry_create.  Errors as there, plus
 * INVALID_ARG for a non-finite offset.
 */
cbct_status cbct_geometry_create_ex(double sad_mm, double sdd_mm,
                                    const double *h_angles_rad, int n_angles,
                                    int nu, int nv, double du_mm, double dv_mm, double off_u_mm, double off_v_mm,
                                    int nx, int ny, int nz, double hx_mm, double hy_mm, double hz_mm,
                                    cbct_geometry **out);

/* Frees the handle, its coarse-level handles and all scratch.  NULL is allowed.  Synchronises the device.  Every pointer
 * obtained from cbct_geometry_coarsen on this handle (or on its coarse levels) is dangling afterwards. */
void cbct_geometry_destroy(cbct_geometry *g);

/* Writes {n_angles, nu, nv, nx, ny, nz} to h_dims6 and {du, dv, hx, hy, hz} to h_sizes5 (either may be NULL). */
cbct_status cbct_geometry_query(const cbct_geometry *g, int *h_dims6, double *h_sizes5);

/*
 * Next-coarser multigrid level ("multi-grid method"; reading O6/Q11): every axis whose spacing
 * is <= sqrt(2) * min(hx,hy,hz) is coarsened by 2 (dims halve, spacing doubles); the detector is
 * binned 2x2 (pitch doubles) iff both x and y were coarsened.  The returned handle is OWNED BY `g`
 * (freed with it, or earlier by a cbct_set_detector_binning call that changes the choice: do not keep the pointer across
 * either; repeated calls return the same handle until then).  h_flags4 (may be NULL) receives
 * {x coarsened, y coarsened, z coarsened, detector binned}.
 * Errors: SHAPE for an odd dimension on an axis that must coarsen (or odd nu/nv when binning).
 */
cbct_status cbct_geometry_coarsen(const cbct_geometry *g, cbct_geometry **out_coarse, int *h_flags4);

/*
 * NEXT-3 (reading Q20): whether the coarse multigrid levels bin the detector 2x2 (on = 1, the default, O6) or keep the
 * detector and the data at full resolution (on = 0).  Changing the choice drops the handle's existing coarse levels
 * (synchronises the device); they are rebuilt on demand.  Applies to every cascade / V-cycle run on this handle.
 * INVALIDATES every coarse-level pointer cbct_geometry_coarsen has returned for this handle and for its coarse levels (the
 * whole chain is freed): using one afterwards is a use-after-free.  Call cbct_geometry_coarsen again to get the new level.
 * A call that does not change the choice frees nothing.
 */
cbct_status cbct_set_detector_binning(cbct_geometry *g, int on);

/*
 * a1. Forward projection q = P f (definition O1): for every angle and detector pixel,
 * the sum over voxels of (length of the segment source->pixel-centre inside the voxel box) * f.
 * Rays that miss the volume give 0.  d_proj is overwritten.
 */
cbct_status cbct_forward(const cbct_geometry *g, const float *d_vol, float *d_proj, void *cuda_stream);

/*
 * Which projector kernel cbct_forward and the cascades use on this handle (and its coarse levels): 0 (default) the march that
 * reads the padded volume copies through the L1 cache, 1 the same march fed by TMA-staged shared-memory bricks (falls back
 * to 0 where a brick would not fit).  Same rays, same arithmetic, same results to rounding order; see DESIGN.md for the
 * measured comparison.
 */
cbct_status cbct_set_projector_staging(cbct_geometry *g, int on);

/*
 * a3. Backprojection G = P^T y — the exact transpose of cbct_forward's matrix ("P^T denotes a
 * matrix transpose"; O2), evaluated as a race-free gather (the paper's "memory conflict" remark,
 * P:95): <P x, y> = <x, P^T y> up to fp32 rounding.  d_vol is overwritten.
 */
cbct_status cbct_backproject(const cbct_geometry *g, const float *d_proj, float *d_vol, void *cuda_stream);

/*
 * Whether the projector and the exact backprojector may use the symmetries of the scan: on = 1 (the default) lets a thread
 *   - march ray (u, v) together with its mirror image (u, nv-1-v) about the central plane z = 0, and gather a voxel row k together
 *     with its mirror image nz-1-k, from one evaluation of the z arithmetic, wherever the geometry is its own mirror image (nz
 *     even, no detector shift in v; the projector also needs nv even);
 *   - march, in addition, the half-turn twins of those rays (angle a + n_angles/2, same pixel, voxels point-reflected about the
 *     rotation axis) from the same ray arithmetic, wherever angles[a + n_angles/2] = angles[a] + pi for every a < n_angles/2
 *     (the second-half rays are then marched from their twin's table entries: an equally good fp32 rounding of the same ray);
 * on = 0 forces the plain kernels.  Same matrix entries either way (O1); results equal to fp32 rounding.  Applies to this
 * handle and its coarse levels.
 */
cbct_status cbct_set_mirror_symmetry(cbct_geometry *g, int on);

/*
 * NEXT-1. The paper's own voxel-driven backprojector, eq. 2, without its prefactor 2/(N_theta A):
 *   (B r)(x) = sum_theta L^3(u*,v*) / (L0 l^2(x)) r(u*,v*)
 * x the voxel centre, (u*,v*) where the line source -> x meets the imager, L0 = sdd, l = |x - S|,
 * L = |(u*,v*) - S|; r is interpolated bilinearly between pixel centres and is 0 outside the detector.
 * It is NOT the transpose of cbct_forward; (du dv / dV) P^T r tends to B r as the grids are refined.
 * d_vol is overwritten.
 */
cbct_status cbct_backproject_eq2(const cbct_geometry *g, const float *d_proj, float *d_vol, void *cuda_stream);

/*
 * Which backprojector step 1 of cbct_fbs_reconstruct uses: the exact transpose (default; the path
 * BASELINE.json's north_star names) or eq. 2 as the paper ran it, g = f - (mu V / beta) (2/(N_theta A)) B r.
 * Applies to this handle and the coarse levels of its cascades.  Errors: INVALID_ARG for another value.
 */
#define CBCT_BACKPROJECTOR_EXACT 0
#define CBCT_BACKPROJECTOR_EQ2 1
cbct_status cbct_set_backprojector(cbct_geometry *g, int mode);

/*
 * a5. TV-prox inner descent (P:89 step 2, "solved by a simple gradient descent method"; O4):
 * n_inner Jacobi steps  u <- u - dt [ beta (u - g) + grad TV_eps(u) ],
 *   dt = omega / (beta + 4 (1/hx^2 + 1/hy^2 + 1/hz^2) / eps),
 * TV_eps = sum sqrt(dx^2+dy^2+dz^2+eps^2) with forward differences divided by the spacing, zero at
 * the far faces.  d_u holds the start on entry and the result on exit (d_u == d_g is NOT allowed;
 * copy g into u to start from g).  Only the volume dims / voxel sizes of `g` are used.
 * Errors: INVALID_ARG if beta < 0, eps <= 0, omega <= 0 or n_inner < 0.
 */
cbct_status cbct_tv_prox(const cbct_geometry *g, const float *d_g, float *d_u,
                         float beta, float eps, float omega, int n_inner, void *cuda_stream);

/*
 * a7. Multigrid transfers between `fine` and its coarse level (cbct_geometry_coarsen(fine)); O6.
 *   cbct_prolong : coarse volume -> fine volume, cell-centred linear interpolation along every
 *                  coarsened axis (fine 2I = 3/4 c[I] + 1/4 c[I-1], fine 2I+1 = 3/4 c[I] + 1/4 c[I+1],
 *                  indices clamped), copy along the others.
 *   cbct_restrict: fine volume -> coarse volume, mean of the children (used for a caller's f0).
 *   cbct_bin2x2  : fine projections -> coarse projections, mean of each 2x2 pixel block (plain
 *                  copy if the level does not bin the detector).
 */
cbct_status cbct_prolong (const cbct_geometry *fine, const float *d_coarse_vol, float *d_fine_vol, void *cuda_stream);
cbct_status cbct_restrict(const cbct_geometry *fine, const float *d_fine_vol, float *d_coarse_vol, void *cuda_stream);
cbct_status cbct_bin2x2  (const cbct_geometry *fine, const float *d_fine_proj, float *d_coarse_proj, void *cuda_stream);

/*
 * Discrete energy of eq. 1 (O3):
 *   E_eps(f) = (1/N_vox) sum n_ijk + mu (1/(N_theta N_pix)) sum (P f - Y)^2 .
 * h_out3 receives {E_eps, E1_eps = TV_eps/N_vox, E2 = data term without mu} as doubles.
 * Runs a forward projection and deterministic two-stage reductions; SYNCHRONISES the stream.
 */
cbct_status cbct_energy(const cbct_geometry *g, const float *d_f, const float *d_Y,
                        float mu, float eps, double *h_out3, void *cuda_stream);

/*
 * The TV term of that energy for callers that must not allocate device memory (O3):
 *   *d_out = TV_eps(f) = sum over voxels of sqrt(dx^2 + dy^2 + dz^2 + eps^2)      (E1_eps of cbct_energy = *d_out / N_vox)
 * with the same differences, fp32 terms and fp64 accumulation as cbct_energy; the two agree to the rounding of the fp64 sums.
 * Who this is for: cbct_energy keeps its per-block partial sums in scratch that the handle obtains with cudaMalloc, and a handle
 * cannot even be created without cudaMalloc.  A host application that has given the whole card to its own memory pool, a monitor
 * running beside a reconstruction that fills HBM on purpose, or a loop that cannot afford the device-wide stall of an
 * allocation cannot use either.  This call needs no handle and allocates nothing, on the device or on the host (no cudaMalloc,
 * cudaFree, events or library routine that allocates): the partial sums go to a fixed 128 KiB array that is part of the
 * library image (every GPU on which the library is loaded carries it until the process exits, used or not).
 *   d_f                 DEVICE, nz*ny*nx floats (x fastest), read only
 *   nx..nz, hx..hz      volume dims and voxel size in mm; no geometry handle is involved
 *   d_out               DEVICE, one double, overwritten; caller-owned like d_f
 * Limit: nx*ny*nz <= 134 217 728 (= 512^3, the largest volume in BASELINE.json) and each dim <= 16384; larger volumes return
 * CBCT_ERR_SHAPE with a message and launch nothing.  INVALID_ARG for NULL pointers, non-positive dims or spacings, eps < 0.
 * Asynchronous on cuda_stream; nothing is synchronised.
 * First call on a device: with that device current, the call looks up the device address of the array once
 * (cudaGetSymbolAddress) and remembers it per device ordinal; make this first call before any stream capture begins.
 * Sharing: there is ONE array per GPU, used by every call from every thread and stream, and it keeps the previous call's
 * partial sums.  No part of it has to start at zero (each call writes every slot it later reads), but two calls that overlap
 * on the GPU - issued on different streams, from one host thread or several - race on it and may both return garbage.  Order
 * such calls on one stream or with events.  (Separate processes have separate copies of the array.)
 */
cbct_status cbct_tv_value_noalloc(const float *d_f, int nx, int ny, int nz, double hx_mm, double hy_mm, double hz_mm,
                                  float eps, double *d_out, void *cuda_stream);

/*
 * The hot path: Algorithm A1 inside a coarse-to-fine cascade (O5/O6).
 * For level l = n_levels-1 (coarsest) ... 0 (finest = g), n_outer_per_level[] listed COARSEST FIRST:
 *   repeat n_outer times:
 *     r = P f - Y                     (a1 + a2, fused)
 *     G = P^T r                       (a3)
 *     gv = f - c G, c = 2 step N_vox / (N_theta N_pix)      (a4; P:87 with eq. 2's factor 2)
 *     u = gv; n_tv_inner TV-prox steps with beta = mu / step  (a5)
 *     f = max(u, 0)                   (a6)
 *   prolong f to the next finer level (a7).
 * Y for the coarse levels is the 2x2-binned d_Y.  d_f0 == NULL starts from zeros; otherwise d_f0 is
 * a FINEST-level volume that is restricted down to the coarsest level.  n_levels == 1 is plain A1.
 * d_f_out (finest level) is overwritten; it may equal d_f0.
 * h_energy_trace: NULL, or sum(n_outer_per_level) doubles receiving E_eps after every outer
 * iteration (costs one extra forward projection and a stream synchronise per iteration).
 * Without a trace the call is asynchronous.
 * Errors: INVALID_ARG for n_levels < 1, negative counts, step <= 0, mu <= 0, eps <= 0, omega <= 0;
 * SHAPE as for cbct_geometry_coarsen.
 */
cbct_status cbct_fbs_reconstruct(const cbct_geometry *g, const float *d_Y, const float *d_f0,
                                 int n_levels, const int *n_outer_per_level, int n_tv_inner,
                                 float step, float mu, float eps, float omega,
                                 float *d_f_out, double *h_energy_trace, void *cuda_stream);

/*
 * NEXT-2. The same cascade with the paper's "Repeat ... until convergence" read as a stopping rule:
 * a level stops after the first outer iteration whose update satisfies
 *   || f_new - f_old ||_2 <= rel_tol || f_new ||_2        (sums accumulated in fp64 on the device),
 * or after n_outer_max_per_level[] iterations (COARSEST FIRST).  rel_tol == 0 is cbct_fbs_reconstruct.
 * h_iters_per_level: NULL, or n_levels ints receiving the iterations run per level (coarsest first).
 * Synchronises the stream once per outer iteration when rel_tol > 0.
 */
cbct_status cbct_fbs_reconstruct_until(const cbct_geometry *g, const float *d_Y, const float *d_f0,
                                       int n_levels, const int *n_outer_max_per_level, int n_tv_inner,
                                       float step, float mu, float eps, float omega, float rel_tol,
                                       float *d_f_out, int *h_iters_per_level, void *cuda_stream);

/*
 * NEXT-3 (reading Q21). FAS V-cycles around Algorithm A1 ("multi-grid method", ref. 20 at P:170 is Brandt; the paper
 * gives no details).  Level l carries F_l(f) = TV_eps(f) + mu'_l ||P_l f - Y_l||^2, mu'_l = mu N_vox,l / (N_theta N_pix,l)
 * (= N_vox,l times the energy of eq. 1).  One cycle on level l with right-hand side tau (0 on the finest level):
 *     nu_pre iterations of A1 on F_l - <tau, .>   (step 1 becomes gv = f - c G + tau / beta)
 *     f_H0 = R f;  tau_H = grad F_{l+1}(f_H0) - R (grad F_l(f) - tau);  f_H = cycle(l+1, f_H0, tau_H)
 *     f = max(f + Prolong(f_H - f_H0), 0);  nu_post iterations of A1 on F_l - <tau, .>
 * and nu_coarse iterations at the coarsest level.  R = mean of the children (cbct_restrict), Prolong = cbct_prolong,
 * Y on the coarse levels as in cbct_fbs_reconstruct.  n_cycles cycles start from d_f0 (NULL = zeros); n_levels == 1 is
 * n_cycles * nu_coarse iterations of plain A1.  d_f_out (finest level) may equal d_f0.
 * h_energy_trace: NULL or n_cycles doubles receiving E_eps after every cycle (synchronises per cycle).
 * Errors: INVALID_ARG for n_levels < 1, negative counts, step/mu/eps/omega <= 0; SHAPE as for cbct_geometry_coarsen.
 */
cbct_status cbct_fbs_vcycle(const cbct_geometry *g, const float *d_Y, const float *d_f0,
                            int n_levels, int n_cycles, int nu_pre, int nu_post, int nu_coarse, int n_tv_inner,
                            float step, float mu, float eps, float omega,
                            float *d_f_out, double *h_energy_trace, void *cuda_stream);

/*
 * NEXT-4. The FDK reconstruction the paper compares against (Feldkamp-Davis-Kress, ref. 1 at P:147; Fig. 1(d) P:105,
 * Fig. 2), reading Q22: d_vol = (pi/N_theta) sum_theta SAD^2/U^2 q_theta(u*,v*) with q the cosine-weighted
 * (SDD/sqrt(SDD^2+u^2+v^2)) projections filtered along u by the band-limited ramp kernel at pitch du SAD/SDD, U the distance
 * of the voxel from the source along the central ray, bilinear interpolation, zero outside the detector (detector positions
 * in fp64, weights and sums in fp32).  Valid for equally spaced views over a full rotation only (no short-scan or half-fan
 * redundancy weights, no apodisation): the angle list must be angles[0] +- 2 pi a / n_angles to 1e-6 of a step, in list order;
 * any other list (a 200 degree arc, a list with a gap or a repeated view) is refused.  A panel shift (cbct_geometry_create_ex) is
 * applied as such: right for a slightly miscentred panel that still sees the whole object, NOT for a half-fan scan, which
 * needs the redundancy weights this routine does not have.  d_vol is overwritten.
 * Errors: SHAPE if the views are not equally spaced over a full turn, or if nu > 8533 (the filter keeps a zero-padded fp64
 * row in shared memory).
 */
cbct_status cbct_fdk_reconstruct(const cbct_geometry *g, const float *d_Y, float *d_vol, void *cuda_stream);

/*
 * NEXT-4. The two halves of one outer iteration of A1, for drivers that put an exchange step between them: with
 * the angle list partitioned over several GPUs (one handle per GPU holding its share of the angles and of d_Y),
 * every GPU computes its partial data gradient, the partial volumes are summed (one all-reduce), and every GPU
 * applies the same prox step.  P^T over a subset of the angles is an exact partial sum of the full P^T.
 *   cbct_data_gradient : d_G = P^T (P d_f - d_Y) over this handle's angles (with CBCT_BACKPROJECTOR_EQ2:
 *                        (dV/(du dv)) B (P d_f - d_Y)).  d_G is overwritten; must not alias d_f.
 *   cbct_prox_step     : d_f_out = max(0, TVprox(d_f - c d_G)), n_inner steps with beta, eps, omega as in
 *                        cbct_tv_prox; c = 2 step N_vox / (N_theta N_pix) with the TOTAL number of angles.
 *                        d_f_out may alias d_f, not d_G.
 */
cbct_status cbct_data_gradient(const cbct_geometry *g, const float *d_f, const float *d_Y, float *d_G, void *cuda_stream);
cbct_status cbct_prox_step(const cbct_geometry *g, const float *d_f, const float *d_G, float c, float beta,
                           float eps, float omega, int n_inner, float *d_f_out, void *cuda_stream);

/*
 * NEXT-4. The angle-sharded cascade itself: this handle holds THIS RANK'S share of the views and d_Y_local
 * their data; every rank holds the whole volume.  Per outer iteration: cbct_data_gradient -> `allreduce` (sum of the gradient
 * volume over the ranks, in place) -> cbct_prox_step with c = 2 step N_vox / (n_angles_total N_pix), inside the same
 * coarse-to-fine cascade as cbct_fbs_reconstruct (n_outer_per_level COARSEST FIRST, d_f0 NULL = zeros).
 *   allreduce(d_buf, count, user, cuda_stream): must sum d_buf[0..count) over all ranks in place, ordered on cuda_stream
 *     (e.g. ncclAllReduce, or torch.distributed.all_reduce on the tensor that owns d_buf); returns 0 on success.
 *     NULL = single rank (the result then equals cbct_fbs_reconstruct).
 *   d_G_scratch: caller-owned device buffer of nx*ny*nz floats — the buffer handed to `allreduce` (its first N_vox,l floats
 *     on level l), so the caller knows which of its tensors is exchanged.  Must not alias d_f_out.
 * Errors: INVALID_ARG (NULL, bad counts, n_angles_total < this handle's views, callback failure), SHAPE as for coarsen.
 */
typedef int (*cbct_allreduce_fn)(float *d_buf, unsigned long long count, void *user, void *cuda_stream);
cbct_status cbct_fbs_reconstruct_sharded(const cbct_geometry *g, const float *d_Y_local, const float *d_f0,
                                         int n_levels, const int *n_outer_per_level, int n_tv_inner,
                                         float step, float mu, float eps, float omega, int n_angles_total,
                                         cbct_allreduce_fn allreduce, void *user, float *d_G_scratch,
                                         float *d_f_out, void *cuda_stream);

/*
 * The order of operations of that cascade, as a routine over callbacks (host logic only, makes no CUDA call): used by
 * cbct_fbs_reconstruct_sharded with this library's operators, and callable with any other operators that keep the
 * per-level state themselves (the CPU multi-rank tests drive it with the fp64 oracle over gloo).  Every callback returns
 * 0 on success (a cbct_status value is passed through).  Levels: 0 = finest ... n_levels-1 = coarsest.
 *   level_sizes(user, l, &n_vox, &n_pix)   sizes of level l (n_pix = nu*nv of that level)
 *   bin(user, l)                           Y_{l+1} = 2x2-binned Y_l
 *   start(user, L, have_f0)                f_L = 0, or the caller's f0 restricted level by level down to L
 *   data_gradient(user, l)                 G_l = P^T (P f_l - Y_l) over this rank's views
 *   all_reduce(user, l)                    G_l summed over the ranks (may be NULL: single rank)
 *   prox_step(user, l, c, beta)            f_l = max(0, TVprox(f_l - c G_l))
 *   prolong(user, l)                       f_{l-1} = Prolong f_l
 * with c = 2 step N_vox,l / (n_angles_total N_pix,l) and beta = mu / step.
 */
typedef struct cbct_cascade_ops {
    void *user;
    int (*level_sizes)(void *user, int level, unsigned long long *n_vox, unsigned long long *n_pix);
    int (*bin)(void *user, int level);
    int (*start)(void *user, int coarsest_level, int have_f0);
    int (*data_gradient)(void *user, int level);
    int (*all_reduce)(void *user, int level);
    int (*prox_step)(void *user, int level, double c, double beta);
    int (*prolong)(void *user, int level);
} cbct_cascade_ops;
cbct_status cbct_cascade_run(const cbct_cascade_ops *ops, int n_levels, const int *n_outer_per_level,
                             double step, double mu, int n_angles_total, int have_f0);

/*
 * Host-buffer variants (end-to-end path): same operations with HOST pointers; each call copies its
 * inputs host->device and its result device->host on `cuda_stream` (use pinned host memory for
 * full copy speed) and returns after synchronising the stream.  cbct_fbs_reconstruct_host uploads h_Y from an internal
 * second stream, behind h_f0 on the bus and beside the cascade's first kernels (those that do not need Y); its result equals
 * cbct_fbs_reconstruct on the same data bit for bit.
 */
cbct_status cbct_forward_host(const cbct_geometry *g, const float *h_vol, float *h_proj, void *cuda_stream);
cbct_status cbct_backproject_host(const cbct_geometry *g, const float *h_proj, float *h_vol, void *cuda_stream);
cbct_status cbct_tv_prox_host(const cbct_geometry *g, const float *h_g, float *h_u,
                              float beta, float eps, float omega, int n_inner, void *cuda_stream);
cbct_status cbct_fbs_reconstruct_host(const cbct_geometry *g, const float *h_Y, const float *h_f0,
                                      int n_levels, const int *n_outer_per_level, int n_tv_inner,
                                      float step, float mu, float eps, float omega,
                                      float *h_f_out, double *h_energy_trace, void *cuda_stream);

/*
 * Per-kernel-class device timing (CUDA events recorded around each launch on the launching stream).
 * Classes: 0 pad/transposed volume copies, 1 forward projector, 2 projection scaling + prefix sums along v, 3 backprojector
 * gather, 4 combine / gradient step, 5 TV sweep, 6 multigrid transfers, 7 reductions.
 * cbct_profile_read fills h_ms[CBCT_PROFILE_TAGS] (summed milliseconds) and h_count[] (launch groups)
 * since the last reset; it waits for the recorded events.  Off by default.
 */
#define CBCT_PROFILE_TAGS 8
cbct_status cbct_profile_enable(int on);
cbct_status cbct_profile_read(double *h_ms, unsigned long long *h_count, int reset);

/* Number of kernels this library has launched in this process so far (monotone counter). */
unsigned long long cbct_launch_count(void);

/* Bytes of device memory currently held by the handle (tables + scratch, all levels). */
unsigned long long cbct_device_bytes(const cbct_geometry *g);

/*
 * Debugging aid standing in for a memory checker: after cbct_set_guard_mode(1) every device buffer that a handle allocates
 * (tables at creation, scratch on first use) is placed between two 4096-byte regions filled with a pattern (slower: every
 * allocation synchronises the device).  cbct_check_guards synchronises the device and writes to *h_bad_bytes the number of
 * pattern bytes around the buffers of this handle and of its coarse levels that no longer hold the pattern: 0 unless a kernel
 * wrote outside a library-owned buffer.  Process-wide switch; affects allocations made after the call.
 */
cbct_status cbct_set_guard_mode(int on);
cbct_status cbct_check_guards(const cbct_geometry *g, unsigned long long *h_bad_bytes);

/* Description of the last failure on this host thread ("" if none).  Static storage. */
const char *cbct_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* CBCT_H */
