// NEXT-3: FAS V-cycles around Algorithm A1 ("we employed the well developed multi-grid method", ref. 20 = Brandt at
// P:170; the paper gives no details: reading Q21 of DESIGN.md).  Host-side driver only: every arithmetic step runs in the
// kernels of the hot path (projector, gather, TV sweeps, transfers) plus tv_grad_kernel.
//
// Level l has the objective F_l(f) = N_vox,l E_eps,l(f) = TV_eps,l(f) + mu'_l ||P_l f - Y_l||^2, mu'_l = mu N_vox,l/(N_theta N_pix,l);
// grad F_l discretises the level-independent functional derivative V dE/df, so it moves between levels by averaging.
//   V(l, f, tau):  f <- nu_pre iterations of A1 on F_l - <tau, .>
//                  f_H0 = R f;  tau_H = grad F_{l+1}(f_H0) - R (grad F_l(f) - tau);  f_H = V(l+1, f_H0, tau_H)
//                  f <- max(f + Prolong(f_H - f_H0), 0);  f <- nu_post iterations of A1 on F_l - <tau, .>
// with nu_coarse iterations at the coarsest level; R = mean of the children, Prolong = the cascade's interpolation.
#include <vector>

#include "cbct_internal.h"

namespace {
struct VCtx {
    std::vector<cbct_geometry *> lev;
    std::vector<const float *> Y;
    int n_levels, nu_pre, nu_post, nu_coarse, n_inner;
    float step, mu, eps, omega;
    cudaStream_t st;
};

// d_out = grad F_l(f) - tau  (tau may be NULL).  Uses lev->vc_e as scratch for grad TV.
cbct_status grad_objective(VCtx &c, int l, const float *f, const float *tau, float *d_out)
{
    cbct_geometry *g = c.lev[l];
    CBCT_TRY(ensure(g, &g->vc_e, g->n_vox()));
    CBCT_TRY(op_data_gradient(g, f, c.Y[l], d_out, c.st));                            // P^T (P f - Y)
    CBCT_TRY(op_tv_grad(g, f, c.eps, g->vc_e, c.st));
    const float mu2 = (float)(2.0 * (double)c.mu * (double)g->n_vox() / ((double)g->na * g->nu * g->nv));
    CBCT_TRY(op_axpy_clamp(g, g->vc_e, d_out, -mu2, 0, d_out, c.st));                 // grad TV + 2 mu' P^T r
    if (tau) CBCT_TRY(op_axpy_clamp(g, d_out, tau, 1.f, 0, d_out, c.st));             // - tau
    return CBCT_OK;
}

cbct_status smooth(VCtx &c, int l, float *f, const float *tau, int n)
{
    return op_fbs_level(c.lev[l], c.Y[l], f, n, c.n_inner, c.step, c.mu, c.eps, c.omega, nullptr, 0.f, nullptr, tau, c.st);
}

cbct_status vcycle(VCtx &c, int l, float *f, const float *tau)
{
    if (l == c.n_levels - 1) return smooth(c, l, f, tau, c.nu_coarse);
    cbct_geometry *g = c.lev[l], *gc = c.lev[l + 1];
    CBCT_TRY(smooth(c, l, f, tau, c.nu_pre));
    CBCT_TRY(ensure(g, &g->vc_d, g->n_vox()));
    CBCT_TRY(ensure(gc, &gc->vc_tau, gc->n_vox()));
    CBCT_TRY(ensure(gc, &gc->vc_f0, gc->n_vox()));
    CBCT_TRY(ensure(gc, &gc->vol_f, gc->n_vox()));
    CBCT_TRY(ensure(gc, &gc->vc_d, gc->n_vox()));
    CBCT_TRY(grad_objective(c, l, f, tau, g->vc_d));                                  // D = grad F_l(f) - tau
    CBCT_TRY(op_restrict(g, f, gc->vc_f0, c.st));                                     // f_H0 = R f
    CBCT_TRY(op_restrict(g, g->vc_d, gc->vc_d, c.st));                                // R D
    CBCT_TRY(grad_objective(c, l + 1, gc->vc_f0, gc->vc_d, gc->vc_tau));              // tau_H = grad F_H(f_H0) - R D
    CBCT_CUDA(cudaMemcpyAsync(gc->vol_f, gc->vc_f0, gc->n_vox() * sizeof(float), cudaMemcpyDeviceToDevice, c.st));
    CBCT_TRY(vcycle(c, l + 1, gc->vol_f, gc->vc_tau));
    CBCT_TRY(op_axpy_clamp(gc, gc->vol_f, gc->vc_f0, 1.f, 0, gc->vc_d, c.st));        // e_H = f_H - f_H0
    CBCT_TRY(op_prolong(g, gc->vc_d, g->vc_d, c.st));
    CBCT_TRY(op_axpy_clamp(g, f, g->vc_d, -1.f, 1, f, c.st));                         // f = max(f + Prolong e_H, 0)
    return smooth(c, l, f, tau, c.nu_post);
}
}  // namespace

extern "C" cbct_status cbct_fbs_vcycle(const cbct_geometry *gc, const float *d_Y, const float *d_f0, int n_levels, int n_cycles,
                                       int nu_pre, int nu_post, int nu_coarse, int n_tv_inner, float step, float mu, float eps,
                                       float omega, float *d_f_out, double *h_energy_trace, void *stream)
{
    if (!gc || !d_Y || !d_f_out) { cbct_set_error("cbct_fbs_vcycle: NULL argument"); return CBCT_ERR_INVALID_ARG; }
    if (n_levels < 1 || n_levels > 16 || n_cycles < 0 || nu_pre < 0 || nu_post < 0 || nu_coarse < 0 || n_tv_inner < 0 ||
        !(step > 0.f) || !(mu > 0.f) || !(eps > 0.f) || !(omega > 0.f)) {
        cbct_set_error("cbct_fbs_vcycle: n_levels < 1 (or > 16), a negative count, or step, mu, eps, omega not > 0");
        return CBCT_ERR_INVALID_ARG;
    }
    VCtx c;
    c.n_levels = n_levels; c.nu_pre = nu_pre; c.nu_post = nu_post; c.nu_coarse = nu_coarse; c.n_inner = n_tv_inner;
    c.step = step; c.mu = mu; c.eps = eps; c.omega = omega; c.st = (cudaStream_t)stream;
    c.lev.resize(n_levels);
    c.Y.resize(n_levels);
    c.lev[0] = const_cast<cbct_geometry *>(gc);
    c.Y[0] = d_Y;
    for (int l = 1; l < n_levels; ++l) {
        CBCT_TRY(cbct_geometry_coarsen(c.lev[l - 1], &c.lev[l], nullptr));
        CBCT_TRY(ensure(c.lev[l], &c.lev[l]->Y_level, c.lev[l]->n_proj()));
        CBCT_TRY(op_bin2x2(c.lev[l - 1], c.Y[l - 1], c.lev[l]->Y_level, c.st));
        c.Y[l] = c.lev[l]->Y_level;
    }
    const size_t bytes = c.lev[0]->n_vox() * sizeof(float);
    if (!d_f0) CBCT_CUDA(cudaMemsetAsync(d_f_out, 0, bytes, c.st));
    else if (d_f0 != d_f_out) CBCT_CUDA(cudaMemcpyAsync(d_f_out, d_f0, bytes, cudaMemcpyDeviceToDevice, c.st));
    for (int n = 0; n < n_cycles; ++n) {
        CBCT_TRY(vcycle(c, 0, d_f_out, nullptr));
        if (h_energy_trace) {
            double e3[3];
            CBCT_TRY(op_energy(c.lev[0], d_f_out, d_Y, mu, eps, e3, c.st));
            h_energy_trace[n] = e3[0];
        }
    }
    return CBCT_OK;
}
