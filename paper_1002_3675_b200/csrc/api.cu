// C-ABI entry points (include/cbct.h): argument checks, scratch, the FBS / multigrid driver (L2) and
// the host-buffer variants.  All arithmetic of the hot path runs in the kernels of projector.cu,
// backprojector.cu, tv.cu and transfers.cu.
#include <cmath>
#include <vector>

#include "cbct_internal.h"

#define REQUIRE(cond, ...)                                  \
    do {                                                    \
        if (!(cond)) {                                      \
            cbct_set_error(__VA_ARGS__);                    \
            return CBCT_ERR_INVALID_ARG;                    \
        }                                                   \
    } while (0)

static inline cbct_geometry *mut(const cbct_geometry *g) { return const_cast<cbct_geometry *>(g); }

extern "C" cbct_status cbct_forward(const cbct_geometry *gc, const float *d_vol, float *d_proj, void *stream)
{
    REQUIRE(gc && d_vol && d_proj, "cbct_forward: NULL argument");
    cbct_geometry *g = mut(gc);
    cudaStream_t st = (cudaStream_t)stream;
    CBCT_TRY(op_pad_copies(g, d_vol, st));
    return op_forward_padded(g, d_proj, nullptr, 0, st);
}

extern "C" cbct_status cbct_backproject(const cbct_geometry *gc, const float *d_proj, float *d_vol, void *stream)
{
    REQUIRE(gc && d_proj && d_vol, "cbct_backproject: NULL argument");
    cbct_geometry *g = mut(gc);
    cudaStream_t st = (cudaStream_t)stream;
    CBCT_TRY(ensure_zeroed(g, &g->proj_tmp, g->n_proj(), st));
    CBCT_TRY(op_backproject_prefix(g, d_proj, 1, g->proj_tmp, st));       // l * y and its prefix sums along v
    CBCT_TRY(op_backproject_gather(g, g->proj_tmp, st));
    return op_combine(g, nullptr, 0.f, 0, d_vol, st);
}

extern "C" cbct_status cbct_backproject_eq2(const cbct_geometry *gc, const float *d_proj, float *d_vol, void *stream)
{
    REQUIRE(gc && d_proj && d_vol, "cbct_backproject_eq2: NULL argument");
    return op_backproject_eq2(mut(gc), d_proj, nullptr, 0.f, 0, d_vol, (cudaStream_t)stream);
}

extern "C" cbct_status cbct_set_backprojector(cbct_geometry *g, int mode)
{
    REQUIRE(g, "cbct_set_backprojector: NULL handle");
    REQUIRE(mode == CBCT_BACKPROJECTOR_EXACT || mode == CBCT_BACKPROJECTOR_EQ2, "cbct_set_backprojector: unknown mode %d", mode);
    for (cbct_geometry *q = g; q; q = q->coarse) q->bp_mode = mode;      // coarse levels created later inherit it (cbct_geometry_coarsen)
    return CBCT_OK;
}

extern "C" cbct_status cbct_set_projector_staging(cbct_geometry *g, int on)
{
    REQUIRE(g, "cbct_set_projector_staging: NULL handle");
    for (cbct_geometry *q = g; q; q = q->coarse) q->fw_staged = on != 0;
    return CBCT_OK;
}

extern "C" cbct_status cbct_set_mirror_symmetry(cbct_geometry *g, int on)
{
    REQUIRE(g, "cbct_set_mirror_symmetry: NULL handle");
    for (cbct_geometry *q = g; q; q = q->coarse) q->use_mirror = on != 0;
    return CBCT_OK;
}

static float tv_dt(const cbct_geometry *g, float beta, float eps, float omega)
{
    const double K = 4.0 * (1.0 / (g->hx * g->hx) + 1.0 / (g->hy * g->hy) + 1.0 / (g->hz * g->hz));
    return (float)((double)omega / ((double)beta + K / (double)eps));
}

// n_inner Jacobi steps starting from u_start (may alias gv or u_out); the result ends in u_out.
// vol_b is the second ping-pong buffer.  clamp_last fuses a6 into the last step's store.
static cbct_status tv_inner(cbct_geometry *g, const float *gv, const float *u_start, float *u_out, float beta,
                            float eps, float omega, int n_inner, int clamp_last, cudaStream_t st)
{
    const size_t bytes = g->n_vox() * sizeof(float);
    if (n_inner == 0) {
        if (u_start != u_out) CBCT_CUDA(cudaMemcpyAsync(u_out, u_start, bytes, cudaMemcpyDeviceToDevice, st));
        return CBCT_OK;
    }
    CBCT_TRY(ensure(g, &g->vol_b, g->n_vox()));
    const float dt = tv_dt(g, beta, eps, omega);
    const float *src = u_start;
    for (int m = 0; m < n_inner; ++m) {
        float *dst = ((n_inner - 1 - m) % 2 == 0) ? u_out : g->vol_b;     // the last step lands in u_out
        if (src == dst) {                                                  // only m == 0 with u_start == u_out
            CBCT_CUDA(cudaMemcpyAsync(g->vol_b, src, bytes, cudaMemcpyDeviceToDevice, st));
            src = g->vol_b;
        }
        CBCT_TRY(op_tv_sweep(g, src, gv, dst, beta, eps, dt, clamp_last && m == n_inner - 1, st));
        src = dst;
    }
    return CBCT_OK;
}

extern "C" cbct_status cbct_tv_prox(const cbct_geometry *gc, const float *d_g, float *d_u, float beta, float eps,
                                    float omega, int n_inner, void *stream)
{
    REQUIRE(gc && d_g && d_u, "cbct_tv_prox: NULL argument");
    REQUIRE(d_g != d_u, "cbct_tv_prox: d_u must not alias d_g");
    REQUIRE(beta >= 0.f && eps > 0.f && omega > 0.f && n_inner >= 0, "cbct_tv_prox: beta < 0, eps <= 0, omega <= 0 or n_inner < 0");
    return tv_inner(mut(gc), d_g, d_u, d_u, beta, eps, omega, n_inner, 0, (cudaStream_t)stream);
}

extern "C" cbct_status cbct_prolong(const cbct_geometry *fine, const float *c, float *f, void *stream)
{
    REQUIRE(fine && c && f, "cbct_prolong: NULL argument");
    return op_prolong(mut(fine), c, f, (cudaStream_t)stream);
}
extern "C" cbct_status cbct_restrict(const cbct_geometry *fine, const float *f, float *c, void *stream)
{
    REQUIRE(fine && c && f, "cbct_restrict: NULL argument");
    return op_restrict(mut(fine), f, c, (cudaStream_t)stream);
}
extern "C" cbct_status cbct_bin2x2(const cbct_geometry *fine, const float *y, float *yc, void *stream)
{
    REQUIRE(fine && y && yc, "cbct_bin2x2: NULL argument");
    return op_bin2x2(mut(fine), y, yc, (cudaStream_t)stream);
}

// E_eps(f); synchronises.
cbct_status op_energy(cbct_geometry *g, const float *d_f, const float *d_Y, float mu, float eps,
                               double *out3, cudaStream_t st)
{
    CBCT_TRY(ensure_zeroed(g, &g->proj_tmp, g->n_proj(), st));
    CBCT_TRY(ensure(g, &g->red_out, (size_t)2));
    if (!g->h_red) CBCT_CUDA(cudaMallocHost((void **)&g->h_red, 2 * sizeof(double)));
    CBCT_TRY(op_pad_copies(g, d_f, st));
    CBCT_TRY(op_forward_padded(g, g->proj_tmp, nullptr, 0, st));
    CBCT_TRY(op_sumsq_diff(g, g->proj_tmp, d_Y, g->n_proj(), g->red_out + 0, st));
    CBCT_TRY(op_tv_value(g, d_f, eps, g->red_out + 1, st));
    CBCT_CUDA(cudaMemcpyAsync(g->h_red, g->red_out, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CBCT_CUDA(cudaStreamSynchronize(st));
    const double e2 = g->h_red[0] / ((double)g->na * g->nu * g->nv);
    const double e1 = g->h_red[1] / (double)g->n_vox();
    out3[0] = e1 + (double)mu * e2;
    out3[1] = e1;
    out3[2] = e2;
    return CBCT_OK;
}

extern "C" cbct_status cbct_energy(const cbct_geometry *gc, const float *d_f, const float *d_Y, float mu, float eps,
                                   double *h_out3, void *stream)
{
    REQUIRE(gc && d_f && d_Y && h_out3, "cbct_energy: NULL argument");
    REQUIRE(eps >= 0.f, "cbct_energy: eps < 0");
    return op_energy(mut(gc), d_f, d_Y, mu, eps, h_out3, (cudaStream_t)stream);
}

// ---- the two halves of an outer iteration, for drivers that put an exchange step between them (NEXT-4) ----
extern "C" cbct_status cbct_data_gradient(const cbct_geometry *gc, const float *d_f, const float *d_Y, float *d_G, void *stream)
{
    REQUIRE(gc && d_f && d_Y && d_G, "cbct_data_gradient: NULL argument");
    return op_data_gradient(mut(gc), d_f, d_Y, d_G, (cudaStream_t)stream);
}

cbct_status op_data_gradient(cbct_geometry *g, const float *d_f, const float *d_Y, float *d_G, cudaStream_t st)
{
    CBCT_TRY(ensure_zeroed(g, &g->proj_tmp, g->n_proj(), st));
    CBCT_TRY(op_pad_copies(g, d_f, st));
    if (g->bp_mode == CBCT_BACKPROJECTOR_EQ2) {
        CBCT_TRY(op_forward_padded(g, g->proj_tmp, d_Y, 2, st));
        CBCT_TRY(ensure(g, &g->vol_a, g->n_vox()));
        CBCT_CUDA(cudaMemsetAsync(g->vol_a, 0, g->n_vox() * sizeof(float), st));
        // 0 - (-(dV/(du dv))) B r
        return op_backproject_eq2(g, g->proj_tmp, g->vol_a, -(float)((g->hx * g->hy * g->hz) / (g->du * g->dv)), 0, d_G, st);
    }
    CBCT_TRY(op_forward_padded(g, g->proj_tmp, d_Y, 1, st));
    CBCT_TRY(op_backproject_prefix(g, g->proj_tmp, 0, nullptr, st));
    CBCT_TRY(op_backproject_gather(g, g->proj_tmp, st));
    return op_combine(g, nullptr, 0.f, 0, d_G, st);
}

extern "C" cbct_status cbct_prox_step(const cbct_geometry *gc, const float *d_f, const float *d_G, float c, float beta,
                                      float eps, float omega, int n_inner, float *d_f_out, void *stream)
{
    REQUIRE(gc && d_f && d_G && d_f_out, "cbct_prox_step: NULL argument");
    REQUIRE(beta >= 0.f && eps > 0.f && omega > 0.f && n_inner >= 0, "cbct_prox_step: beta < 0, eps <= 0, omega <= 0 or n_inner < 0");
    REQUIRE(d_G != d_f_out, "cbct_prox_step: d_f_out must not alias d_G");
    cbct_geometry *g = mut(gc);
    cudaStream_t st = (cudaStream_t)stream;
    CBCT_TRY(ensure(g, &g->vol_a, g->n_vox()));
    CBCT_TRY(op_axpy_clamp(g, d_f, d_G, c, n_inner == 0, g->vol_a, st));        // gv = f - c G (clamped if no TV step follows)
    if (n_inner == 0) {
        CBCT_CUDA(cudaMemcpyAsync(d_f_out, g->vol_a, g->n_vox() * sizeof(float), cudaMemcpyDeviceToDevice, st));
        return CBCT_OK;
    }
    return tv_inner(g, g->vol_a, g->vol_a, d_f_out, beta, eps, omega, n_inner, 1, st);
}

// One level of Algorithm A1: f (in/out, level-sized device buffer).
// rel_tol > 0: stop after the first iteration with ||f_new - f_old||_2 <= rel_tol ||f_new||_2 (NEXT-2; sums in fp64,
// one stream synchronise per iteration); *iters receives the number of iterations run.
// tau != nullptr (FAS coarse problems, vcycle.cu): the linear term -<tau, f> joins the gradient of step 1, gv = f - c G + tau / beta.
cbct_status op_fbs_level(cbct_geometry *g, const float *d_Y, float *f, int n_outer, int n_inner, float step,
                         float mu, float eps, float omega, double *trace, float rel_tol, int *iters, const float *tau,
                         cudaStream_t st, const std::function<cbct_status()> *y_gate)
{
    if (rel_tol > 0.f) {
        CBCT_TRY(ensure(g, &g->vol_c, g->n_vox()));
        CBCT_TRY(ensure(g, &g->red_out, (size_t)2));
        if (!g->h_red) CBCT_CUDA(cudaMallocHost((void **)&g->h_red, 2 * sizeof(double)));
    }
    if (iters) *iters = 0;
    CBCT_TRY(ensure_zeroed(g, &g->proj_tmp, g->n_proj(), st));
    CBCT_TRY(ensure(g, &g->vol_a, g->n_vox()));
    const float beta = mu / step;
    const float c = (float)(2.0 * (double)step * (double)g->n_vox() / ((double)g->na * g->nu * g->nv));
    // one outer iteration (steps 1-3 of A1) on stream s: the same launches with the same arguments every iteration
    // gate != nullptr (host-buffer path, first iteration only): Y is still on its way to the device, so the projection runs
    // without the fused residual, then the gate waits for Y (and bins it for the coarse levels), then a2 runs on its own
    auto iteration = [&](cudaStream_t s, const std::function<cbct_status()> *gate) -> cbct_status {
        CBCT_TRY(op_pad_copies(g, f, s));
        if (g->bp_mode == CBCT_BACKPROJECTOR_EQ2) {
            // the paper's step 1 (P:87 with eq. 2): dE2/df = (2/(N_theta A)) B r, so gv = f - c (dV/(du dv)) B r
            const float c2 = (float)((double)c * (g->hx * g->hy * g->hz) / (g->du * g->dv));
            if (gate) {
                CBCT_TRY(op_forward_padded(g, g->proj_tmp, nullptr, 0, s));
                CBCT_TRY((*gate)());
                CBCT_TRY(op_residual(g, g->proj_tmp, d_Y, 2, s));
            } else
                CBCT_TRY(op_forward_padded(g, g->proj_tmp, d_Y, 2, s));  // P f - Y              a1+a2
            CBCT_TRY(op_backproject_eq2(g, g->proj_tmp, f, c2, n_inner == 0 && !tau, g->vol_a, s));   // a3 (eq. 2) + a4 (+ a6)
            if (tau) CBCT_TRY(op_axpy_clamp(g, g->vol_a, tau, -1.f / beta, n_inner == 0, g->vol_a, s));
            if (n_inner == 0) CBCT_CUDA(cudaMemcpyAsync(f, g->vol_a, g->n_vox() * sizeof(float), cudaMemcpyDeviceToDevice, s));
            else CBCT_TRY(tv_inner(g, g->vol_a, g->vol_a, f, beta, eps, omega, n_inner, 1, s));
        } else {
            if (gate) {
                CBCT_TRY(op_forward_padded(g, g->proj_tmp, nullptr, 0, s));
                CBCT_TRY((*gate)());
                CBCT_TRY(op_residual(g, g->proj_tmp, d_Y, 1, s));
            } else
                CBCT_TRY(op_forward_padded(g, g->proj_tmp, d_Y, 1, s));      // l (P f - Y)          a1+a2
            CBCT_TRY(op_backproject_prefix(g, g->proj_tmp, 0, nullptr, s));
            CBCT_TRY(op_backproject_gather(g, g->proj_tmp, s));              // P^T (P f - Y)        a3
            CBCT_TRY(op_combine(g, f, c, n_inner == 0 && !tau, g->vol_a, s));    // gv = f - c G (a4), clamped (a6) if nothing follows
            if (tau) CBCT_TRY(op_axpy_clamp(g, g->vol_a, tau, -1.f / beta, n_inner == 0, g->vol_a, s));   // + tau / beta
            if (n_inner == 0) CBCT_CUDA(cudaMemcpyAsync(f, g->vol_a, g->n_vox() * sizeof(float), cudaMemcpyDeviceToDevice, s));
            else CBCT_TRY(tv_inner(g, g->vol_a, g->vol_a, f, beta, eps, omega, n_inner, 1, s));   // u0 = gv (Q7); a5 + a6
        }
        return CBCT_OK;
    };
    // Small volumes are launch-bound (c1: a dozen kernels of 5-10 us per iteration): after one eager iteration (which makes
    // every allocation) the iteration is captured once into a CUDA graph on an internal stream and replayed on the caller's.
    // Any failure to capture falls back to eager launches.
    struct GraphExecGuard {                                      // destroyed on every way out of this function, error returns included
        cudaGraphExec_t e = nullptr;
        ~GraphExecGuard() { if (e) cudaGraphExecDestroy(e); }
    } guard;
    cudaGraphExec_t &gexec = guard.e;
    const bool want_graph = !trace && rel_tol == 0.f && !y_gate && !cbct_profile_is_on() && n_outer >= 6 && g->n_vox() <= ((size_t)1 << 20);
    for (int it = 0; it < n_outer; ++it) {
        if (rel_tol > 0.f) CBCT_CUDA(cudaMemcpyAsync(g->vol_c, f, g->n_vox() * sizeof(float), cudaMemcpyDeviceToDevice, st));
        if (want_graph && it == 1 && !gexec) {
            if (!g->graph_stream && cudaStreamCreateWithFlags(&g->graph_stream, cudaStreamNonBlocking) != cudaSuccess) g->graph_stream = nullptr;
            cudaGraph_t graph = nullptr;
            if (g->graph_stream && cudaStreamBeginCapture(g->graph_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
                const unsigned long long n0 = g_cbct_launches.load();
                const cbct_status cs = iteration(g->graph_stream, nullptr);  // recorded, not run
                g_cbct_launches.store(n0);
                const cudaError_t ce = cudaStreamEndCapture(g->graph_stream, &graph);
                if (cs != CBCT_OK || ce != cudaSuccess || !graph || cudaGraphInstantiate(&gexec, graph, 0) != cudaSuccess) gexec = nullptr;
                if (graph) cudaGraphDestroy(graph);
            }
            (void)cudaGetLastError();                            // a failed capture leaves no sticky error behind
        }
        if (gexec && it >= 1) {
            CBCT_CUDA(cudaGraphLaunch(gexec, st));
            g_cbct_launches += g->launches_per_iteration;
        } else {
            const unsigned long long n0 = g_cbct_launches.load();
            CBCT_TRY(iteration(st, it == 0 ? y_gate : nullptr));
            g->launches_per_iteration = g_cbct_launches.load() - n0;
        }
        if (trace) {
            double e3[3];
            CBCT_TRY(op_energy(g, f, d_Y, mu, eps, e3, st));
            trace[it] = e3[0];
        }
        if (iters) *iters = it + 1;
        if (rel_tol > 0.f) {
            CBCT_TRY(op_sumsq_diff(g, f, g->vol_c, g->n_vox(), g->red_out + 0, st));
            CBCT_TRY(op_sumsq_diff(g, f, nullptr, g->n_vox(), g->red_out + 1, st));
            CBCT_CUDA(cudaMemcpyAsync(g->h_red, g->red_out, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
            CBCT_CUDA(cudaStreamSynchronize(st));
            if (std::sqrt(g->h_red[0]) <= (double)rel_tol * std::sqrt(g->h_red[1])) break;
        }
    }
    return CBCT_OK;
}

static cbct_status fbs_cascade(const cbct_geometry *gc, const float *d_Y, const float *d_f0, int n_levels,
                               const int *n_outer, int n_inner, float step, float mu, float eps, float omega,
                               float *d_f_out, double *trace, float rel_tol, int *iters_per_level, void *stream,
                               cudaEvent_t y_ready = nullptr)
{
    REQUIRE(gc && d_Y && d_f_out && n_outer, "cbct_fbs_reconstruct: NULL argument");
    REQUIRE(n_levels >= 1 && n_levels <= 16 && n_inner >= 0, "cbct_fbs_reconstruct: n_levels < 1 (or > 16) or n_tv_inner < 0");
    REQUIRE(step > 0.f && mu > 0.f && eps > 0.f && omega > 0.f, "cbct_fbs_reconstruct: step, mu, eps and omega must be > 0");
    for (int l = 0; l < n_levels; ++l) REQUIRE(n_outer[l] >= 0, "cbct_fbs_reconstruct: negative iteration count");
    cudaStream_t st = (cudaStream_t)stream;

    // level handles, finest first
    std::vector<cbct_geometry *> lev(n_levels);
    lev[0] = mut(gc);
    for (int l = 1; l < n_levels; ++l) {
        CBCT_TRY(cbct_geometry_coarsen(lev[l - 1], &lev[l], nullptr));
    }

    // data per level: level 0 uses d_Y, coarser levels their own binned copy.  y_ready (host-buffer path): d_Y is still being
    // uploaded on another stream; everything that does not need it (the restriction of f0, the padded copies and the first
    // projection of the coarsest level) runs first, then `gate` waits for the upload and bins
    std::vector<const float *> Y(n_levels);
    Y[0] = d_Y;
    for (int l = 1; l < n_levels; ++l) {
        CBCT_TRY(ensure(lev[l], &lev[l]->Y_level, lev[l]->n_proj()));
        Y[l] = lev[l]->Y_level;
    }
    bool y_here = false;
    const std::function<cbct_status()> gate = [&]() -> cbct_status {
        if (y_here) return CBCT_OK;
        y_here = true;
        if (y_ready) CBCT_CUDA(cudaStreamWaitEvent(st, y_ready, 0));
        for (int l = 1; l < n_levels; ++l) CBCT_TRY(op_bin2x2(lev[l - 1], Y[l - 1], lev[l]->Y_level, st));
        return CBCT_OK;
    };
    if (!y_ready) CBCT_TRY(gate());
    // current iterate per level lives in vol_f of that level (level 0: the caller's output buffer)
    std::vector<float *> F(n_levels);
    F[0] = d_f_out;
    for (int l = 1; l < n_levels; ++l) {
        CBCT_TRY(ensure(lev[l], &lev[l]->vol_f, lev[l]->n_vox()));
        F[l] = lev[l]->vol_f;
    }
    // start: zeros, or the caller's fine f0 restricted down
    const int L = n_levels - 1;
    if (!d_f0) {
        CBCT_CUDA(cudaMemsetAsync(F[L], 0, lev[L]->n_vox() * sizeof(float), st));
    } else {
        if (d_f0 != d_f_out)
            CBCT_CUDA(cudaMemcpyAsync(F[0], d_f0, lev[0]->n_vox() * sizeof(float), cudaMemcpyDeviceToDevice, st));
        for (int l = 1; l < n_levels; ++l) CBCT_TRY(op_restrict(lev[l - 1], F[l - 1], F[l], st));
    }
    int done = 0;
    for (int l = L; l >= 0; --l) {
        const int n = n_outer[L - l];
        CBCT_TRY(op_fbs_level(lev[l], Y[l], F[l], n, n_inner, step, mu, eps, omega, trace ? trace + done : nullptr, rel_tol,
                              iters_per_level ? iters_per_level + (L - l) : nullptr, nullptr, st, y_here ? nullptr : &gate));
        CBCT_TRY(gate());                                        // a level with no iterations has not opened it
        done += n;
        if (l > 0) CBCT_TRY(op_prolong(lev[l - 1], F[l], F[l - 1], st));
    }
    return CBCT_OK;
}

extern "C" cbct_status cbct_fbs_reconstruct(const cbct_geometry *gc, const float *d_Y, const float *d_f0, int n_levels,
                                            const int *n_outer, int n_inner, float step, float mu, float eps,
                                            float omega, float *d_f_out, double *trace, void *stream)
{
    return fbs_cascade(gc, d_Y, d_f0, n_levels, n_outer, n_inner, step, mu, eps, omega, d_f_out, trace, 0.f, nullptr, stream);
}

extern "C" cbct_status cbct_fbs_reconstruct_until(const cbct_geometry *gc, const float *d_Y, const float *d_f0, int n_levels,
                                                  const int *n_outer_max, int n_inner, float step, float mu, float eps,
                                                  float omega, float rel_tol, float *d_f_out, int *h_iters_per_level,
                                                  void *stream)
{
    REQUIRE(rel_tol >= 0.f, "cbct_fbs_reconstruct_until: rel_tol < 0");
    return fbs_cascade(gc, d_Y, d_f0, n_levels, n_outer_max, n_inner, step, mu, eps, omega, d_f_out, nullptr, rel_tol,
                       h_iters_per_level, stream);
}

// ---- host-buffer variants ----------------------------------------------------------------------
extern "C" cbct_status cbct_forward_host(const cbct_geometry *gc, const float *h_vol, float *h_proj, void *stream)
{
    REQUIRE(gc && h_vol && h_proj, "cbct_forward_host: NULL argument");
    cbct_geometry *g = mut(gc);
    cudaStream_t st = (cudaStream_t)stream;
    CBCT_TRY(ensure(g, &g->host_stage_vol, g->n_vox()));
    CBCT_TRY(ensure(g, &g->host_stage_proj, g->n_proj()));
    CBCT_CUDA(cudaMemcpyAsync(g->host_stage_vol, h_vol, g->n_vox() * sizeof(float), cudaMemcpyHostToDevice, st));
    CBCT_TRY(cbct_forward(g, g->host_stage_vol, g->host_stage_proj, stream));
    CBCT_CUDA(cudaMemcpyAsync(h_proj, g->host_stage_proj, g->n_proj() * sizeof(float), cudaMemcpyDeviceToHost, st));
    CBCT_CUDA(cudaStreamSynchronize(st));
    return CBCT_OK;
}

extern "C" cbct_status cbct_backproject_host(const cbct_geometry *gc, const float *h_proj, float *h_vol, void *stream)
{
    REQUIRE(gc && h_vol && h_proj, "cbct_backproject_host: NULL argument");
    cbct_geometry *g = mut(gc);
    cudaStream_t st = (cudaStream_t)stream;
    CBCT_TRY(ensure(g, &g->host_stage_vol, g->n_vox()));
    CBCT_TRY(ensure(g, &g->host_stage_proj, g->n_proj()));
    CBCT_CUDA(cudaMemcpyAsync(g->host_stage_proj, h_proj, g->n_proj() * sizeof(float), cudaMemcpyHostToDevice, st));
    CBCT_TRY(cbct_backproject(g, g->host_stage_proj, g->host_stage_vol, stream));
    CBCT_CUDA(cudaMemcpyAsync(h_vol, g->host_stage_vol, g->n_vox() * sizeof(float), cudaMemcpyDeviceToHost, st));
    CBCT_CUDA(cudaStreamSynchronize(st));
    return CBCT_OK;
}

extern "C" cbct_status cbct_tv_prox_host(const cbct_geometry *gc, const float *h_g, float *h_u, float beta, float eps,
                                         float omega, int n_inner, void *stream)
{
    REQUIRE(gc && h_g && h_u, "cbct_tv_prox_host: NULL argument");
    cbct_geometry *g = mut(gc);
    cudaStream_t st = (cudaStream_t)stream;
    CBCT_TRY(ensure(g, &g->host_stage_vol, g->n_vox()));
    CBCT_TRY(ensure(g, &g->host_stage_vol2, g->n_vox()));
    CBCT_CUDA(cudaMemcpyAsync(g->host_stage_vol, h_g, g->n_vox() * sizeof(float), cudaMemcpyHostToDevice, st));
    CBCT_CUDA(cudaMemcpyAsync(g->host_stage_vol2, h_u, g->n_vox() * sizeof(float), cudaMemcpyHostToDevice, st));
    CBCT_TRY(cbct_tv_prox(g, g->host_stage_vol, g->host_stage_vol2, beta, eps, omega, n_inner, stream));
    CBCT_CUDA(cudaMemcpyAsync(h_u, g->host_stage_vol2, g->n_vox() * sizeof(float), cudaMemcpyDeviceToHost, st));
    CBCT_CUDA(cudaStreamSynchronize(st));
    return CBCT_OK;
}

extern "C" cbct_status cbct_fbs_reconstruct_host(const cbct_geometry *gc, const float *h_Y, const float *h_f0,
                                                 int n_levels, const int *n_outer, int n_inner, float step, float mu,
                                                 float eps, float omega, float *h_f_out, double *trace, void *stream)
{
    REQUIRE(gc && h_Y && h_f_out, "cbct_fbs_reconstruct_host: NULL argument");
    cbct_geometry *g = mut(gc);
    cudaStream_t st = (cudaStream_t)stream;
    CBCT_TRY(ensure(g, &g->host_stage_vol, g->n_vox()));
    CBCT_TRY(ensure(g, &g->host_stage_proj, g->n_proj()));
    if (!g->copy_stream) {
        CBCT_CUDA(cudaStreamCreateWithFlags(&g->copy_stream, cudaStreamNonBlocking));
        CBCT_CUDA(cudaEventCreateWithFlags(&g->ev_f0, cudaEventDisableTiming));
        CBCT_CUDA(cudaEventCreateWithFlags(&g->ev_Y, cudaEventDisableTiming));
    }
    // The cascade needs all of f0 before its first kernel (the coarsest level starts from the restricted f0), Y only when the
    // first projection of that level is done: f0 goes first, on the caller's stream; Y follows it on the bus from a second
    // stream (behind an event, so that the two uploads do not share the bandwidth) while the restriction, the padded copies and
    // that projection run; the cascade waits for Y where it first needs it.  The download of f cannot be hidden.
    if (h_f0)
        CBCT_CUDA(cudaMemcpyAsync(g->host_stage_vol, h_f0, g->n_vox() * sizeof(float), cudaMemcpyHostToDevice, st));
    CBCT_CUDA(cudaEventRecord(g->ev_f0, st));
    CBCT_CUDA(cudaStreamWaitEvent(g->copy_stream, g->ev_f0, 0));
    CBCT_CUDA(cudaMemcpyAsync(g->host_stage_proj, h_Y, g->n_proj() * sizeof(float), cudaMemcpyHostToDevice, g->copy_stream));
    CBCT_CUDA(cudaEventRecord(g->ev_Y, g->copy_stream));
    const cbct_status rc = fbs_cascade(g, g->host_stage_proj, h_f0 ? g->host_stage_vol : nullptr, n_levels, n_outer, n_inner, step,
                                       mu, eps, omega, g->host_stage_vol, trace, 0.f, nullptr, stream, g->ev_Y);
    if (rc != CBCT_OK) {                                         // never leave the upload running into a buffer the caller may free
        cudaStreamSynchronize(g->copy_stream);
        return rc;
    }
    CBCT_CUDA(cudaMemcpyAsync(h_f_out, g->host_stage_vol, g->n_vox() * sizeof(float), cudaMemcpyDeviceToHost, st));
    CBCT_CUDA(cudaStreamSynchronize(st));
    return CBCT_OK;
}
