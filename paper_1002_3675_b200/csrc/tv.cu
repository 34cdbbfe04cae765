// a5/a6: one Jacobi step of the TV-prox inner descent (P:89 step 2; O4 in DESIGN.md), with the
// non-negativity clamp fused into the last step's store.
//
//   u' = u - dt [ beta (u - g) + grad TV_eps(u) ],
//   grad TV_eps(u)[ijk] = -(qx+qy+qz)|ijk + qx|i-1 + qy|j-1 + qz|k-1,   q_a = (d_a / h_a) / n,
//   d_a forward difference / h_a (0 at the far face), n = sqrt(dx^2+dy^2+dz^2+eps^2).
//
// HBM-bound (12 B/voxel: read u, read g, write u').  A CTA stages a 32x8x8 tile of u plus a
// one-voxel halo in shared memory with 16-byte loads, computes the three fluxes q once per site
// (one rsqrt per site instead of four per voxel) into shared memory, then writes the update.
#include "cbct_internal.h"

namespace {
constexpr int TX = 32, TY = 8, TZ = 8;
constexpr int SUX = 40;                       // su row: [3] = x0-1 halo, [4..35] interior, [36] = x0+32 halo
constexpr int NSITE = (TX + 1) * (TY + 1) * (TZ + 1);

__device__ __forceinline__ float inv_sqrt_nr(float x)
{
    float y = rsqrtf(x);
    return y * fmaf(-0.5f * x, y * y, 1.5f);      // one Newton step: ~1 ulp
}

__global__ void __launch_bounds__(256)
tv_sweep_kernel(const float *__restrict__ u_in, const float *__restrict__ gv, float *__restrict__ u_out,
                int nx, int ny, int nz, float ihx, float ihy, float ihz, float beta, float eps2, float dt,
                int clamp, int vec_ok)
{
    __shared__ __align__(16) float su[TZ + 2][TY + 2][SUX];
    __shared__ float sq[3][NSITE];
    const int tid = threadIdx.x;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = blockIdx.z * TZ;
    const size_t sxy = (size_t)nx * ny;

    // ---- stage u (interior: 4 rows x 8 float4 per warp instruction) ----
    {
        const int warp = tid >> 5, lane = tid & 31;
        const int rsub = lane >> 3, q = lane & 7;
        for (int row = warp * 4 + rsub; row < (TZ + 2) * (TY + 2); row += 32) {
            const int kz = row / (TY + 2), jy = row % (TY + 2);
            const int gk = z0 + kz - 1, gj = y0 + jy - 1, gi = x0 + 4 * q;
            float4 val = make_float4(0.f, 0.f, 0.f, 0.f);
            if (gk >= 0 && gk < nz && gj >= 0 && gj < ny) {
                const float *src = u_in + (size_t)gk * sxy + (size_t)gj * nx + gi;
                if (vec_ok && gi + 3 < nx) {
                    val = __ldg(reinterpret_cast<const float4 *>(src));
                } else {
                    if (gi < nx) val.x = __ldg(src);
                    if (gi + 1 < nx) val.y = __ldg(src + 1);
                    if (gi + 2 < nx) val.z = __ldg(src + 2);
                    if (gi + 3 < nx) val.w = __ldg(src + 3);
                }
            }
            *reinterpret_cast<float4 *>(&su[kz][jy][4 + 4 * q]) = val;
        }
        // x halos
        for (int h = tid; h < 2 * (TZ + 2) * (TY + 2); h += 256) {
            const int row = h >> 1, side = h & 1;
            const int kz = row / (TY + 2), jy = row % (TY + 2);
            const int gk = z0 + kz - 1, gj = y0 + jy - 1, gi = side ? x0 + TX : x0 - 1;
            float val = 0.f;
            if (gk >= 0 && gk < nz && gj >= 0 && gj < ny && gi >= 0 && gi < nx)
                val = __ldg(u_in + (size_t)gk * sxy + (size_t)gj * nx + gi);
            su[kz][jy][side ? 4 + TX : 3] = val;
        }
    }
    __syncthreads();

    // ---- fluxes at sites (-1..TX-1, -1..TY-1, -1..TZ-1) relative to the tile ----
    for (int s = tid; s < NSITE; s += 256) {
        const int sx = s % (TX + 1), t = s / (TX + 1);
        const int sy = t % (TY + 1), sz = t / (TY + 1);
        const int gi = x0 + sx - 1, gj = y0 + sy - 1, gk = z0 + sz - 1;
        float qx = 0.f, qy = 0.f, qz = 0.f;
        if (gi >= 0 && gj >= 0 && gk >= 0 && gi < nx && gj < ny && gk < nz) {
            const float c = su[sz][sy][sx + 3];
            const float dx = (gi + 1 < nx) ? (su[sz][sy][sx + 4] - c) * ihx : 0.f;
            const float dy = (gj + 1 < ny) ? (su[sz][sy + 1][sx + 3] - c) * ihy : 0.f;
            const float dz = (gk + 1 < nz) ? (su[sz + 1][sy][sx + 3] - c) * ihz : 0.f;
            const float inv = inv_sqrt_nr(fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, eps2))));
            qx = dx * inv * ihx;
            qy = dy * inv * ihy;
            qz = dz * inv * ihz;
        }
        sq[0][s] = qx;
        sq[1][s] = qy;
        sq[2][s] = qz;
    }
    __syncthreads();

    // ---- update ----
    const int tx = tid & 31, ty = tid >> 5;
    const int gi = x0 + tx, gj = y0 + ty;
    if (gi >= nx || gj >= ny) return;
#pragma unroll
    for (int tz = 0; tz < TZ; ++tz) {
        const int gk = z0 + tz;
        if (gk >= nz) break;
        const int s = ((tz + 1) * (TY + 1) + (ty + 1)) * (TX + 1) + (tx + 1);
        const float grad = -(sq[0][s] + sq[1][s] + sq[2][s]) + sq[0][s - 1] + sq[1][s - (TX + 1)] +
                           sq[2][s - (TX + 1) * (TY + 1)];
        const size_t o = (size_t)gk * sxy + (size_t)gj * nx + gi;
        const float u = su[tz + 1][ty + 1][tx + 4];
        float un = u - dt * fmaf(beta, u - __ldg(gv + o), grad);
        if (clamp) un = fmaxf(un, 0.f);
        u_out[o] = un;
    }
}

// TV_eps(f) partial sums (energy monitor): one double per block.
__global__ void __launch_bounds__(256)
tv_value_kernel(const float *__restrict__ f, int nx, int ny, int nz, float ihx, float ihy, float ihz,
                float eps2, double *__restrict__ partial)
{
    const size_t n = (size_t)nx * ny * nz, sxy = (size_t)nx * ny;
    double acc = 0.0;
    for (size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x; o < n; o += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(o % nx), j = (int)((o / nx) % ny), k = (int)(o / sxy);
        const float c = __ldg(f + o);
        const float dx = (i + 1 < nx) ? (__ldg(f + o + 1) - c) * ihx : 0.f;
        const float dy = (j + 1 < ny) ? (__ldg(f + o + nx) - c) * ihy : 0.f;
        const float dz = (k + 1 < nz) ? (__ldg(f + o + sxy) - c) * ihz : 0.f;
        acc += (double)sqrtf(fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, eps2))));
    }
    __shared__ double sh[256];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}

// grad TV_eps(f) itself (O4; the FAS right-hand side of vcycle.cu needs it apart from a descent step): one thread per voxel
// evaluates 1/n at its own site and at the three sites below it with IEEE square roots and divisions (the result feeds a
// difference of two gradients, so it is kept at full fp32 accuracy; this kernel is not on the hot path).
__global__ void __launch_bounds__(256)
tv_grad_kernel(const float *__restrict__ f, float *__restrict__ out, int nx, int ny, int nz, float ihx, float ihy, float ihz, float eps2)
{
    const size_t n = (size_t)nx * ny * nz, sxy = (size_t)nx * ny;
    for (size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x; o < n; o += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(o % nx), j = (int)((o / nx) % ny), k = (int)(o / sxy);
        auto site = [&](size_t s, int si, int sj, int sk, float &qx, float &qy, float &qz) {
            const float c = __ldg(f + s);
            const float dx = (si + 1 < nx) ? (__ldg(f + s + 1) - c) * ihx : 0.f;
            const float dy = (sj + 1 < ny) ? (__ldg(f + s + nx) - c) * ihy : 0.f;
            const float dz = (sk + 1 < nz) ? (__ldg(f + s + sxy) - c) * ihz : 0.f;
            const float inv = 1.f / sqrtf(fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, eps2))));
            qx = dx * inv * ihx; qy = dy * inv * ihy; qz = dz * inv * ihz;
        };
        float qx, qy, qz, t0, t1, t2;
        site(o, i, j, k, qx, qy, qz);
        float grad = -(qx + qy + qz);
        if (i > 0) { site(o - 1, i - 1, j, k, t0, t1, t2); grad += t0; }
        if (j > 0) { site(o - nx, i, j - 1, k, t0, t1, t2); grad += t1; }
        if (k > 0) { site(o - sxy, i, j, k - 1, t0, t1, t2); grad += t2; }
        out[o] = grad;
    }
}

__global__ void final_sum_kernel(const double *__restrict__ partial, int n, double *__restrict__ out)
{
    __shared__ double sh[256];
    double acc = 0.0;
    for (int q = threadIdx.x; q < n; q += 256) acc += partial[q];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = sh[0];
}
}  // namespace

cbct_status op_tv_sweep(cbct_geometry *g, const float *u_in, const float *gv, float *u_out,
                        float beta, float eps, float dt, int clamp, cudaStream_t st)
{
    ProfileScope ps(5, st);
    int done = 0;
#ifndef CBCT_TV_NO_TMA
    CBCT_TRY(op_tv_sweep_tma(g, u_in, gv, u_out, beta, eps, dt, clamp, st, &done));    // nx <= 512, nx % 4 == 0: TMA-fed rows (tv_tma.cu)
    if (done) return CBCT_OK;
#endif
    CBCT_TRY(op_tv_sweep_rows(g, u_in, gv, u_out, beta, eps, dt, clamp, st, &done));   // nx <= 512: row-streaming kernel (tv_rows.cu)
    if (done) return CBCT_OK;
    dim3 grid((g->nx + TX - 1) / TX, (g->ny + TY - 1) / TY, (g->nz + TZ - 1) / TZ);
    const int vec_ok = (g->nx % 4 == 0) && ((reinterpret_cast<uintptr_t>(u_in) & 15) == 0);
    tv_sweep_kernel<<<grid, 256, 0, st>>>(u_in, gv, u_out, g->nx, g->ny, g->nz, (float)(1.0 / g->hx),
                                          (float)(1.0 / g->hy), (float)(1.0 / g->hz), beta, eps * eps, dt,
                                          clamp, vec_ok);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

cbct_status op_tv_grad(cbct_geometry *g, const float *f, float eps, float *out, cudaStream_t st)
{
    ProfileScope ps(5, st);
    const size_t n = g->n_vox();
    const int blocks = (int)((n + 255) / 256 < 148 * 16 ? (n + 255) / 256 : 148 * 16);
    tv_grad_kernel<<<blocks, 256, 0, st>>>(f, out, g->nx, g->ny, g->nz, (float)(1.0 / g->hx), (float)(1.0 / g->hy),
                                           (float)(1.0 / g->hz), eps * eps);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

constexpr int kRedBlocks = 1024;

cbct_status op_tv_value(cbct_geometry *g, const float *f, float eps, double *d_out, cudaStream_t st)
{
    CBCT_TRY(ensure(g, &g->red_partial, (size_t)kRedBlocks));
    ProfileScope ps(7, st);
    tv_value_kernel<<<kRedBlocks, 256, 0, st>>>(f, g->nx, g->ny, g->nz, (float)(1.0 / g->hx), (float)(1.0 / g->hy),
                                                (float)(1.0 / g->hz), eps * eps, g->red_partial);
    CBCT_LAUNCH_CHECK();
    final_sum_kernel<<<1, 256, 0, st>>>(g->red_partial, kRedBlocks, d_out);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

// sum (a - b)^2 (b may be NULL), deterministic two-stage, double accumulation
namespace {
__global__ void __launch_bounds__(256)
sumsq_kernel(const float *__restrict__ a, const float *__restrict__ b, size_t n, double *__restrict__ partial)
{
    double acc = 0.0;
    for (size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x; o < n; o += (size_t)gridDim.x * blockDim.x) {
        const float dlt = b ? __ldg(a + o) - __ldg(b + o) : __ldg(a + o);
        acc += (double)dlt * (double)dlt;
    }
    __shared__ double sh[256];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}
}  // namespace

cbct_status op_sumsq_diff(cbct_geometry *g, const float *a, const float *b, size_t n, double *d_out, cudaStream_t st)
{
    CBCT_TRY(ensure(g, &g->red_partial, (size_t)kRedBlocks));
    ProfileScope ps(7, st);
    sumsq_kernel<<<kRedBlocks, 256, 0, st>>>(a, b, n, g->red_partial);
    CBCT_LAUNCH_CHECK();
    final_sum_kernel<<<1, 256, 0, st>>>(g->red_partial, kRedBlocks, d_out);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}
