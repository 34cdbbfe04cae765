// a5/a6, fast path: the TV-prox Jacobi step of tv.cu for volumes with nx <= 512, streamed along z.
//
// Same arithmetic as tv_sweep_kernel (P:89 step 2; O4 in DESIGN.md):
//   u' = u - dt [ beta (u - g) + grad TV_eps(u) ],  grad TV_eps(u)[ijk] = -(qx+qy+qz)|ijk + qx|i-1 + qy|j-1 + qz|k-1,
//   q_a = (d_a / h_a) / n,  d_a forward difference / h_a (0 at the far face),  n = sqrt(dx^2+dy^2+dz^2+eps^2).
// Layout of the work: a warp owns one whole x row (lane l holds XPT consecutive voxels in registers, so
// the x neighbours are registers or one shuffle), a CTA owns NW consecutive rows y0-1 .. y0+NW-2 and
// marches through a chunk of z planes keeping u(z), u(z+1) and qz(z-1) in registers.  Per plane each
// warp publishes its row of u(z+1) and of qy(z) in shared memory for the neighbouring rows (double
// buffered: one barrier per plane).  The first warp only produces qy for the row below it, the last
// only publishes u for the row above it; the NW-2 rows in between are updated and stored.
// HBM traffic per voxel and step: read u, read g, write u' (12 B), each once, as 16-byte accesses.
// 1/n is one rsqrt.approx (<= 2 ulp): measured against the fp64 oracle the result is the same to 1e-9 with or
// without a Newton step (relative error of 10 sweeps 3e-8, of the update itself 3e-6).

#include "cbct_internal.h"

namespace {

template <int XPT, bool VEC>
__device__ __forceinline__ void load_row(float (&r)[XPT], const float *__restrict__ row, int x0, int nx, bool ok)
{
    if constexpr (VEC) {
#pragma unroll
        for (int q = 0; q < XPT / 4; ++q) {
            float4 t = make_float4(0.f, 0.f, 0.f, 0.f);
            if (ok && x0 + 4 * q < nx) t = __ldg(reinterpret_cast<const float4 *>(row + x0 + 4 * q));
            r[4 * q] = t.x; r[4 * q + 1] = t.y; r[4 * q + 2] = t.z; r[4 * q + 3] = t.w;
        }
    } else {
#pragma unroll
        for (int e = 0; e < XPT; ++e) r[e] = (ok && x0 + e < nx) ? __ldg(row + x0 + e) : 0.f;
    }
}

// shared rows are stored lane-interleaved ([e/4][lane] float4, or [e][lane] floats): writer and reader use the
// same lane, so the format is private to this kernel and free of bank conflicts
template <int XPT>
__device__ __forceinline__ void put_row(float *srow, int lane, const float (&r)[XPT])
{
    if constexpr (XPT % 4 == 0) {
#pragma unroll
        for (int q = 0; q < XPT / 4; ++q)
            reinterpret_cast<float4 *>(srow)[q * 32 + lane] = make_float4(r[4 * q], r[4 * q + 1], r[4 * q + 2], r[4 * q + 3]);
    } else {
#pragma unroll
        for (int e = 0; e < XPT; ++e) srow[e * 32 + lane] = r[e];
    }
}

template <int XPT>
__device__ __forceinline__ void get_row(const float *srow, int lane, float (&r)[XPT])
{
    if constexpr (XPT % 4 == 0) {
#pragma unroll
        for (int q = 0; q < XPT / 4; ++q) {
            const float4 t = reinterpret_cast<const float4 *>(srow)[q * 32 + lane];
            r[4 * q] = t.x; r[4 * q + 1] = t.y; r[4 * q + 2] = t.z; r[4 * q + 3] = t.w;
        }
    } else {
#pragma unroll
        for (int e = 0; e < XPT; ++e) r[e] = srow[e * 32 + lane];
    }
}

template <int XPT, int NW, bool VEC>
__global__ void __launch_bounds__(32 * NW)
tv_rows_kernel(const float *__restrict__ u_in, const float *__restrict__ gv, float *__restrict__ u_out,
               const int nx, const int ny, const int nz, const float ihx2, const float ihy2, const float ihz2,
               const float beta, const float eps2, const float dt, const int clamp, const int zchunk)
{
    constexpr int W = 32 * XPT, ROWS = NW - 2;
    extern __shared__ __align__(16) float sm[];
    float *B = sm;                    // [2][NW][W]  rows of u, plane parity
    float *Q = sm + 2 * NW * W;       // [2][NW][W]  rows of qy, plane parity
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int y = blockIdx.x * ROWS - 1 + w;
    const int zc0 = blockIdx.y * zchunk, zc1 = min(zc0 + zchunk, nz);
    const int x0 = lane * XPT;
    const bool row_ok = y >= 0 && y < ny;
    const bool do_flux = row_ok && w < NW - 1;
    const bool do_upd = row_ok && w >= 1 && w < NW - 1;
    const bool has_yp = y + 1 < ny;
    const size_t sxy = (size_t)nx * ny;
    const size_t rowoff = (size_t)max(y, 0) * nx;

    float uc[XPT], un[XPT], u2[XPT], qzp[XPT];
    const int zs = max(zc0 - 1, 0);
    load_row<XPT, VEC>(uc, u_in + (size_t)zs * sxy + rowoff, x0, nx, row_ok);
    load_row<XPT, VEC>(un, u_in + (size_t)min(zs + 1, nz - 1) * sxy + rowoff, x0, nx, row_ok && zs + 1 < nz);
#pragma unroll
    for (int e = 0; e < XPT; ++e) qzp[e] = 0.f;
    put_row<XPT>(B + ((zs & 1) * NW + w) * W, lane, uc);
    __syncthreads();

    for (int z = zs; z < zc1; ++z) {
        const int cur = z & 1, nxt = cur ^ 1;
        const bool has_zp = z + 1 < nz;
        // plane z+2 is requested now and consumed at the end of this iteration: its latency hides behind the
        // fluxes and the barrier of plane z
        load_row<XPT, VEC>(u2, u_in + (size_t)min(z + 2, nz - 1) * sxy + rowoff, x0, nx, row_ok && z + 2 < nz && z + 1 < zc1);
        put_row<XPT>(B + (nxt * NW + w) * W, lane, un);
        float g[XPT];
        const bool upd = do_upd && z >= zc0;
        if (upd) load_row<XPT, VEC>(g, gv + (size_t)z * sxy + rowoff, x0, nx, true);

        float qx[XPT], qy[XPT], qz[XPT];
        if (do_flux) {
            float uy[XPT];
            get_row<XPT>(B + (cur * NW + w + 1) * W, lane, uy);
            // zero difference at the far faces (uniform per warp / per plane): compare the row with itself
            if (!has_yp) {
#pragma unroll
                for (int e = 0; e < XPT; ++e) uy[e] = uc[e];
            }
            if (!has_zp) {
#pragma unroll
                for (int e = 0; e < XPT; ++e) un[e] = uc[e];
            }
            const float xr_next = __shfl_down_sync(0xffffffffu, uc[0], 1);      // first voxel of the lane to the right
#pragma unroll
            for (int e = 0; e < XPT; ++e) {
                const float c = uc[e];
                const float xr = e + 1 < XPT ? uc[e + 1 < XPT ? e + 1 : 0] : xr_next;
                const float dx = (x0 + e + 1 < nx) ? xr - c : 0.f;
                const float dy = uy[e] - c;
                const float dz = un[e] - c;
                const float ex = dx * ihx2, ey = dy * ihy2, ez = dz * ihz2;          // d_a / h_a^2
                const float inv = rsqrtf(fmaf(dx, ex, fmaf(dy, ey, fmaf(dz, ez, eps2))));
                qx[e] = ex * inv;
                qy[e] = ey * inv;
                qz[e] = ez * inv;
            }
        } else {
#pragma unroll
            for (int e = 0; e < XPT; ++e) { qx[e] = 0.f; qy[e] = 0.f; qz[e] = 0.f; }
        }
        put_row<XPT>(Q + (cur * NW + w) * W, lane, qy);
        __syncthreads();

        if (upd) {                                                              // warp-uniform
            float qym[XPT];
            get_row<XPT>(Q + (cur * NW + w - 1) * W, lane, qym);
            float qxl = __shfl_up_sync(0xffffffffu, qx[XPT - 1], 1);            // last voxel of the lane to the left
            if (lane == 0) qxl = 0.f;
            float out[XPT];
#pragma unroll
            for (int e = 0; e < XPT; ++e) {
                const float qxm = e > 0 ? qx[e > 0 ? e - 1 : 0] : qxl;
                const float grad = -(qx[e] + qy[e] + qz[e]) + qxm + qym[e] + qzp[e];
                const float c = uc[e];
                float v = c - dt * fmaf(beta, c - g[e], grad);
                if (clamp) v = fmaxf(v, 0.f);
                out[e] = v;
            }
            float *dst = u_out + (size_t)z * sxy + rowoff + x0;
            if constexpr (VEC) {
#pragma unroll
                for (int q = 0; q < XPT / 4; ++q)
                    if (x0 + 4 * q < nx)
                        *reinterpret_cast<float4 *>(dst + 4 * q) = make_float4(out[4 * q], out[4 * q + 1], out[4 * q + 2], out[4 * q + 3]);
            } else {
#pragma unroll
                for (int e = 0; e < XPT; ++e)
                    if (x0 + e < nx) dst[e] = out[e];
            }
        }
#pragma unroll
        for (int e = 0; e < XPT; ++e) { qzp[e] = qz[e]; uc[e] = un[e]; un[e] = u2[e]; }
    }
}

template <int XPT, bool VEC>
cbct_status launch_rows(cbct_geometry *g, const float *u_in, const float *gv, float *u_out, float beta, float eps,
                        float dt, int clamp, cudaStream_t st)
{
    // warps per CTA: measured on B200 (more rows amortise the two halo warps, fewer leave room for more CTAs per SM)
#ifndef CBCT_TV_NW
    constexpr int NW = XPT >= 16 ? 6 : 10;
#else
    constexpr int NW = CBCT_TV_NW;
#endif
    constexpr int ROWS = NW - 2;
    auto kern = tv_rows_kernel<XPT, NW, VEC>;
    const size_t smem = (size_t)4 * NW * 32 * XPT * sizeof(float);
    static int slots = 0;                         // CTAs the device holds at once (per instantiation)
    if (!slots) {
        CBCT_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int dev = 0, sms = 0, per_sm = 0;
        CBCT_CUDA(cudaGetDevice(&dev));
        CBCT_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        CBCT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, 32 * NW, smem));
        slots = sms * (per_sm > 0 ? per_sm : 1);
    }
    // z planes per CTA: a chunk of zc planes costs zc + 1 plane iterations (it recomputes the fluxes of the plane
    // below it) and the grid runs in ceil(CTAs / slots) waves: take the chunk that minimises waves x (zc + 1)
    const int ytiles = (g->ny + ROWS - 1) / ROWS;
    int zchunk = 8;
    long best = -1;
    for (int zc = 4; zc <= 64; ++zc) {
        const long ctas = (long)ytiles * ((g->nz + zc - 1) / zc);
        const long cost = ((ctas + slots - 1) / slots) * (zc + 1);
        if (best < 0 || cost < best) { best = cost; zchunk = zc; }
    }
    dim3 grid(ytiles, (g->nz + zchunk - 1) / zchunk);
    const double hx = g->hx, hy = g->hy, hz = g->hz;
    kern<<<grid, 32 * NW, smem, st>>>(u_in, gv, u_out, g->nx, g->ny, g->nz, (float)(1.0 / (hx * hx)), (float)(1.0 / (hy * hy)),
                                      (float)(1.0 / (hz * hz)), beta, eps * eps, dt, clamp, zchunk);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

}  // namespace

// Returns CBCT_OK and sets *done = 1 if the row-streaming kernel took the step, *done = 0 if the caller
// must use the generic tile kernel (nx > 512).
cbct_status op_tv_sweep_rows(cbct_geometry *g, const float *u_in, const float *gv, float *u_out, float beta, float eps,
                             float dt, int clamp, cudaStream_t st, int *done)
{
    *done = 0;
    if (g->nx > 512) return CBCT_OK;
    const bool vec = (g->nx % 4 == 0) && (((uintptr_t)u_in | (uintptr_t)gv | (uintptr_t)u_out) & 15) == 0;
    *done = 1;
    const int nx = g->nx;
    if (nx <= 32) return launch_rows<1, false>(g, u_in, gv, u_out, beta, eps, dt, clamp, st);
    if (nx <= 64) return launch_rows<2, false>(g, u_in, gv, u_out, beta, eps, dt, clamp, st);
    if (nx <= 128) return vec ? launch_rows<4, true>(g, u_in, gv, u_out, beta, eps, dt, clamp, st)
                              : launch_rows<4, false>(g, u_in, gv, u_out, beta, eps, dt, clamp, st);
    if (nx <= 256) return vec ? launch_rows<8, true>(g, u_in, gv, u_out, beta, eps, dt, clamp, st)
                              : launch_rows<8, false>(g, u_in, gv, u_out, beta, eps, dt, clamp, st);
    return vec ? launch_rows<16, true>(g, u_in, gv, u_out, beta, eps, dt, clamp, st)
               : launch_rows<16, false>(g, u_in, gv, u_out, beta, eps, dt, clamp, st);
}
