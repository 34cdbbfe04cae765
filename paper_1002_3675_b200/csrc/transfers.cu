// a7: multigrid transfers of the coarse-to-fine cascade ("multi-grid method"; O6/Q11 in DESIGN.md).
// All HBM-bound pointwise kernels.
#include <algorithm>

#include "cbct_internal.h"

namespace {
// fine[2I] = 3/4 c[I] + 1/4 c[I-1], fine[2I+1] = 3/4 c[I] + 1/4 c[I+1] (clamped) on coarsened axes.
__device__ __forceinline__ void lin_pair(int fine, int ncoarse, bool coarsened, int &i0, int &i1, float &w1)
{
    if (!coarsened) { i0 = fine; i1 = fine; w1 = 0.f; return; }
    i0 = fine >> 1;
    i1 = (fine & 1) ? min(i0 + 1, ncoarse - 1) : max(i0 - 1, 0);
    w1 = 0.25f;
}

__global__ void __launch_bounds__(256)
prolong_kernel(const float *__restrict__ c, float *__restrict__ f, int nx, int ny, int nz,
               int cx, int cy, int cz, int ax, int ay, int az)
{
    // a CTA takes whole (j,k) rows, a few per block, grid-strided: 4 KB of output per row instead of one tiny CTA per row
    const int rows = ny * nz;
    for (int row = blockIdx.x * blockDim.y + threadIdx.y; row < rows; row += gridDim.x * blockDim.y) {
        const int j = row % ny, k = row / ny;
        int j0, j1, k0, k1;
        float wj, wk;
        lin_pair(j, cy, ay, j0, j1, wj);
        lin_pair(k, cz, az, k0, k1, wk);
        auto at = [&](int kk, int jj, int ii) { return __ldg(c + ((size_t)kk * cy + jj) * cx + ii); };
        // the (j, k) part of the interpolation of coarse column ii
        auto col = [&](int ii) {
            const float a0 = fmaf(wj, at(k0, j1, ii), (1.f - wj) * at(k0, j0, ii));
            const float a1 = fmaf(wj, at(k1, j1, ii), (1.f - wj) * at(k1, j0, ii));
            return fmaf(wk, a1, (1.f - wk) * a0);
        };
        float *frow = f + ((size_t)k * ny + j) * nx;
        if (ax && (nx & 1) == 0 && (reinterpret_cast<unsigned long long>(f) & 7ull) == 0) {
            // x coarsened: a thread makes the fine pair (2I, 2I+1) from the coarse columns I-1, I, I+1 (12 loads for two voxels
            // instead of 16) and stores it as one float2
            for (int I = threadIdx.x; I < cx; I += blockDim.x) {
                const float cm = col(max(I - 1, 0)), c0 = col(I), cp = col(min(I + 1, cx - 1));
                *reinterpret_cast<float2 *>(frow + 2 * I) = make_float2(fmaf(0.25f, cm, 0.75f * c0), fmaf(0.25f, cp, 0.75f * c0));
            }
        } else {
            for (int i = threadIdx.x; i < nx; i += blockDim.x) {
                int i0, i1;
                float wi;
                lin_pair(i, cx, ax, i0, i1, wi);
                frow[i] = fmaf(wi, col(i1), (1.f - wi) * col(i0));
            }
        }
    }
}

__global__ void __launch_bounds__(256)
restrict_kernel(const float *__restrict__ f, float *__restrict__ c, int nx, int ny, int cx, int cy, int cz,
                int ax, int ay, int az)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y, k = blockIdx.z;
    if (i >= cx) return;
    const int sx = ax ? 2 : 1, sy = ay ? 2 : 1, sz = az ? 2 : 1;
    float acc = 0.f;
    for (int dk = 0; dk < sz; ++dk)
        for (int dj = 0; dj < sy; ++dj)
            for (int di = 0; di < sx; ++di)
                acc += __ldg(f + ((size_t)(k * sz + dk) * ny + (j * sy + dj)) * nx + (i * sx + di));
    c[((size_t)k * cy + j) * cx + i] = acc / (float)(sx * sy * sz);
}

__global__ void __launch_bounds__(256)
bin2x2_kernel(const float *__restrict__ y, float *__restrict__ yc, int nu, int nv, int cu, int cv)
{
    const int u = blockIdx.x * blockDim.x + threadIdx.x;
    const int v = blockIdx.y, a = blockIdx.z;
    if (u >= cu) return;
    const float *p = y + ((size_t)a * nv + 2 * v) * nu + 2 * u;
    const float2 r0 = __ldg(reinterpret_cast<const float2 *>(p));
    const float2 r1 = __ldg(reinterpret_cast<const float2 *>(p + nu));
    yc[((size_t)a * cv + v) * cu + u] = 0.25f * ((r0.x + r0.y) + (r1.x + r1.y));
}

}  // namespace

static cbct_status need_coarse(cbct_geometry *fine, cbct_geometry **c)
{
    return cbct_geometry_coarsen(fine, c, nullptr);
}

cbct_status op_prolong(cbct_geometry *fine, const float *c, float *f, cudaStream_t st)
{
    cbct_geometry *gc;
    CBCT_TRY(need_coarse(fine, &gc));
    const int *fl = fine->coarsen_flags;
    ProfileScope ps(6, st);
    const int rows = fine->ny * fine->nz;
    prolong_kernel<<<std::min((rows + 3) / 4, 148 * 16), dim3(64, 4), 0, st>>>(c, f, fine->nx, fine->ny, fine->nz, gc->nx, gc->ny, gc->nz, fl[0], fl[1], fl[2]);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

cbct_status op_restrict(cbct_geometry *fine, const float *f, float *c, cudaStream_t st)
{
    cbct_geometry *gc;
    CBCT_TRY(need_coarse(fine, &gc));
    const int *fl = fine->coarsen_flags;
    ProfileScope ps(6, st);
    dim3 grid((gc->nx + 255) / 256, gc->ny, gc->nz);
    restrict_kernel<<<grid, 256, 0, st>>>(f, c, fine->nx, fine->ny, gc->nx, gc->ny, gc->nz, fl[0], fl[1], fl[2]);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

cbct_status op_bin2x2(cbct_geometry *fine, const float *y, float *yc, cudaStream_t st)
{
    cbct_geometry *gc;
    CBCT_TRY(need_coarse(fine, &gc));
    if (!fine->coarsen_flags[3]) {
        CBCT_CUDA(cudaMemcpyAsync(yc, y, fine->n_proj() * sizeof(float), cudaMemcpyDeviceToDevice, st));
        return CBCT_OK;
    }
    ProfileScope ps(6, st);
    dim3 grid((gc->nu + 255) / 256, gc->nv, gc->na);
    bin2x2_kernel<<<grid, 256, 0, st>>>(y, yc, fine->nu, fine->nv, gc->nu, gc->nv);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

// out = f - c G, optionally clamped at 0 (the gradient step a4 on an already summed gradient volume).  out may alias f or G
// (element-wise, so no restrict qualifiers and plain loads).
__global__ void __launch_bounds__(256) axpy_clamp_kernel(const float *f, const float *G, float c, int clamp, float *out, size_t n)
{
    for (size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x; o < n; o += (size_t)gridDim.x * blockDim.x) {
        float v = fmaf(-c, G[o], f[o]);
        if (clamp) v = fmaxf(v, 0.f);
        out[o] = v;
    }
}

cbct_status op_axpy_clamp(cbct_geometry *g, const float *f, const float *G, float c, int clamp, float *out, cudaStream_t st)
{
    ProfileScope ps(4, st);
    const size_t n = g->n_vox();
    const int blocks = (int)std::min<size_t>((n + 255) / 256, 148 * 16);
    axpy_clamp_kernel<<<blocks, 256, 0, st>>>(f, G, c, clamp, out, n);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}
