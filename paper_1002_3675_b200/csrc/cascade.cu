// NEXT-4: Algorithm A1 with the angle list partitioned over ranks, behind the C ABI.
//
// cbct_cascade_run is the host-side order of operations of the coarse-to-fine cascade with an exchange step in every
// outer iteration — level order, c = 2 step N_vox / (N_theta,total N_pix), beta = mu / step — written against a table of
// callbacks, so the very same routine is driven (a) by the CUDA operators of this library in cbct_fbs_reconstruct_sharded
// and (b) on a CPU-only box by the multi-rank tests (oracle operators + gloo), with no second copy of that logic in Python.
// It makes no CUDA call itself.
#include <vector>

#include "cbct_internal.h"

extern "C" cbct_status cbct_cascade_run(const cbct_cascade_ops *ops, int n_levels, const int *n_outer, double step, double mu,
                                        int n_angles_total, int have_f0)
{
    if (!ops || !n_outer || !ops->level_sizes || !ops->bin || !ops->start || !ops->data_gradient || !ops->prox_step || !ops->prolong) {
        cbct_set_error("cbct_cascade_run: NULL argument or callback");
        return CBCT_ERR_INVALID_ARG;
    }
    if (n_levels < 1 || n_levels > 16 || !(step > 0.0) || !(mu > 0.0) || n_angles_total < 1) {
        cbct_set_error("cbct_cascade_run: n_levels < 1 (or > 16), step <= 0, mu <= 0 or n_angles_total < 1");
        return CBCT_ERR_INVALID_ARG;
    }
    for (int l = 0; l < n_levels; ++l)
        if (n_outer[l] < 0) { cbct_set_error("cbct_cascade_run: negative iteration count"); return CBCT_ERR_INVALID_ARG; }
#define CB(call)                                                                                   \
    do {                                                                                           \
        const int rc_ = (call);                                                                    \
        if (rc_ != 0) {                                                                            \
            if (rc_ < 0 || rc_ > CBCT_ERR_CUDA) cbct_set_error("cbct_cascade_run: callback %s failed (%d)", #call, rc_); \
            return rc_ > 0 && rc_ <= CBCT_ERR_CUDA ? (cbct_status)rc_ : CBCT_ERR_INVALID_ARG;     \
        }                                                                                          \
    } while (0)
    const int L = n_levels - 1;
    for (int l = 0; l < L; ++l) CB(ops->bin(ops->user, l));                  // Y_{l+1} = 2x2-binned Y_l (this rank's views)
    CB(ops->start(ops->user, L, have_f0));                                   // zeros, or the caller's f0 restricted down
    const double beta = mu / step;
    for (int l = L; l >= 0; --l) {                                           // coarsest ... finest; n_outer is coarsest first
        unsigned long long n_vox = 0, n_pix = 0;
        CB(ops->level_sizes(ops->user, l, &n_vox, &n_pix));
        const double c = 2.0 * step * (double)n_vox / ((double)n_angles_total * (double)n_pix);    // P:87 with eq. 2's factor 2
        for (int it = 0; it < n_outer[L - l]; ++it) {
            CB(ops->data_gradient(ops->user, l));                            // G = P_r^T (P_r f - Y_r): an exact partial sum
            if (ops->all_reduce) CB(ops->all_reduce(ops->user, l));          // G = sum over ranks: the ONE exchange per iteration
            CB(ops->prox_step(ops->user, l, c, beta));                       // f = max(0, TVprox(f - c G)), identical on every rank
        }
        if (l > 0) CB(ops->prolong(ops->user, l));                           // f_{l-1} = Prolong f_l
    }
#undef CB
    return CBCT_OK;
}

namespace {
struct ShardCtx {
    std::vector<cbct_geometry *> lev;
    std::vector<const float *> Y;
    std::vector<float *> F;
    float *G = nullptr;                      // caller's scratch: the gradient volume that is exchanged
    const float *f0 = nullptr;
    int n_inner = 0;
    float eps = 0.f, omega = 0.f;
    cbct_allreduce_fn allreduce = nullptr;
    void *user = nullptr;
    cudaStream_t st = nullptr;
};

int sh_sizes(void *u, int l, unsigned long long *n_vox, unsigned long long *n_pix)
{
    ShardCtx *c = (ShardCtx *)u;
    *n_vox = c->lev[l]->n_vox();
    *n_pix = (unsigned long long)c->lev[l]->nu * c->lev[l]->nv;
    return 0;
}
int sh_bin(void *u, int l)
{
    ShardCtx *c = (ShardCtx *)u;
    return op_bin2x2(c->lev[l], c->Y[l], c->lev[l + 1]->Y_level, c->st);
}
int sh_start(void *u, int L, int have_f0)
{
    ShardCtx *c = (ShardCtx *)u;
    if (!have_f0) {
        if (cudaMemsetAsync(c->F[L], 0, c->lev[L]->n_vox() * sizeof(float), c->st) != cudaSuccess) return CBCT_ERR_CUDA;
        return 0;
    }
    if (c->f0 != c->F[0] &&
        cudaMemcpyAsync(c->F[0], c->f0, c->lev[0]->n_vox() * sizeof(float), cudaMemcpyDeviceToDevice, c->st) != cudaSuccess)
        return CBCT_ERR_CUDA;
    for (int l = 1; l <= L; ++l) {
        const cbct_status s = op_restrict(c->lev[l - 1], c->F[l - 1], c->F[l], c->st);
        if (s != CBCT_OK) return s;
    }
    return 0;
}
int sh_grad(void *u, int l)
{
    ShardCtx *c = (ShardCtx *)u;
    return op_data_gradient(c->lev[l], c->F[l], c->Y[l], c->G, c->st);
}
int sh_allreduce(void *u, int l)
{
    ShardCtx *c = (ShardCtx *)u;
    const int rc = c->allreduce(c->G, (unsigned long long)c->lev[l]->n_vox(), c->user, (void *)c->st);
    if (rc != 0) cbct_set_error("cbct_fbs_reconstruct_sharded: the all-reduce callback returned %d", rc);
    return rc == 0 ? 0 : CBCT_ERR_INVALID_ARG;
}
int sh_prox(void *u, int l, double cc, double beta)
{
    ShardCtx *c = (ShardCtx *)u;
    return cbct_prox_step(c->lev[l], c->F[l], c->G, (float)cc, (float)beta, c->eps, c->omega, c->n_inner, c->F[l], (void *)c->st);
}
int sh_prolong(void *u, int l)
{
    ShardCtx *c = (ShardCtx *)u;
    return op_prolong(c->lev[l - 1], c->F[l], c->F[l - 1], c->st);
}
}  // namespace

extern "C" cbct_status cbct_fbs_reconstruct_sharded(const cbct_geometry *gc, const float *d_Y_local, const float *d_f0, int n_levels,
                                                    const int *n_outer, int n_tv_inner, float step, float mu, float eps, float omega,
                                                    int n_angles_total, cbct_allreduce_fn allreduce, void *user, float *d_G_scratch,
                                                    float *d_f_out, void *stream)
{
    if (!gc || !d_Y_local || !d_f_out || !n_outer || !d_G_scratch) {
        cbct_set_error("cbct_fbs_reconstruct_sharded: NULL argument");
        return CBCT_ERR_INVALID_ARG;
    }
    if (n_levels < 1 || n_levels > 16 || n_tv_inner < 0 || !(eps > 0.f) || !(omega > 0.f) || n_angles_total < gc->na) {
        cbct_set_error("cbct_fbs_reconstruct_sharded: n_levels < 1 (or > 16), n_tv_inner < 0, eps <= 0, omega <= 0, or fewer total "
                       "angles than this handle holds");
        return CBCT_ERR_INVALID_ARG;
    }
    if (d_G_scratch == d_f_out) { cbct_set_error("cbct_fbs_reconstruct_sharded: d_G_scratch must not alias d_f_out"); return CBCT_ERR_INVALID_ARG; }
    ShardCtx c;
    c.st = (cudaStream_t)stream;
    c.lev.resize(n_levels); c.Y.resize(n_levels); c.F.resize(n_levels);
    c.lev[0] = const_cast<cbct_geometry *>(gc);
    c.Y[0] = d_Y_local;
    c.F[0] = d_f_out;
    for (int l = 1; l < n_levels; ++l) {
        CBCT_TRY(cbct_geometry_coarsen(c.lev[l - 1], &c.lev[l], nullptr));
        CBCT_TRY(ensure(c.lev[l], &c.lev[l]->Y_level, c.lev[l]->n_proj()));
        CBCT_TRY(ensure(c.lev[l], &c.lev[l]->vol_f, c.lev[l]->n_vox()));
        c.Y[l] = c.lev[l]->Y_level;
        c.F[l] = c.lev[l]->vol_f;
    }
    c.G = d_G_scratch; c.f0 = d_f0; c.n_inner = n_tv_inner; c.eps = eps; c.omega = omega; c.allreduce = allreduce; c.user = user;
    cbct_cascade_ops ops;
    ops.user = &c;
    ops.level_sizes = sh_sizes; ops.bin = sh_bin; ops.start = sh_start; ops.data_gradient = sh_grad;
    ops.all_reduce = allreduce ? sh_allreduce : nullptr;
    ops.prox_step = sh_prox; ops.prolong = sh_prolong;
    return cbct_cascade_run(&ops, n_levels, n_outer, (double)step, (double)mu, n_angles_total, d_f0 != nullptr);
}
