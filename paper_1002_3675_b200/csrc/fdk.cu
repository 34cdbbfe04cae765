// NEXT-4: the FDK reconstruction the paper compares against (Feldkamp, Davis, Kress = ref. 1; Fig. 1(d) at P:105,
// Fig. 2 at P:125).  Reading Q22 of DESIGN.md: equally spaced views over a full rotation, no redundancy weights, no window.
//   1. p1 = Y SDD / sqrt(SDD^2 + us^2 + vs^2)                                   (cosine pre-weight, fused into the row load)
//   2. q[n] = D sum_m h[n-m] p1[m],  D = du SAD/SDD,  h[0] = 1/(4 D^2), h[even] = 0, h[odd k] = -1/(pi^2 k^2 D^2)
//   3. f(x) = (pi / N_theta) sum_a SAD^2/U^2 q_a(u*, v*),  U = SAD - (x cos a + y sin a), (u*, v*) = SDD (lat, z)/U, bilinear
#include "cbct_internal.h"

namespace {
// One CTA per detector row (a, v).  The pre-weighted row sits in shared memory with nu zeros on either side, so that the
// symmetric pairs p1[n-k] + p1[n+k] need no bounds test; only odd k carry weight.  Direct convolution: nu^2/2 FMAs per row
// (2e9 for 40 views of 512 x 384), no FFT and no library on the path.  The sum runs in fp64: the ramp filter removes the
// row's mean, so the result is ~100x smaller than its largest terms and an fp32 running sum would lose the 1e-5 bar.
__global__ void __launch_bounds__(256)
fdk_filter_kernel(const DevGeom d, const float *__restrict__ Y, const float *__restrict__ hk, float *__restrict__ q,
                  const float off_u, const float off_v, const float scale0)
{
    extern __shared__ float row[];                         // [3 nu]: zeros | p1 | zeros
    const int v = blockIdx.x, a = blockIdx.y, nu = d.nu;
    const float vs = fmaf((float)v - 0.5f * (float)(d.nv - 1), d.dv, off_v);
    const float *src = Y + ((size_t)a * d.nv + v) * nu;
    for (int m = threadIdx.x; m < nu; m += blockDim.x) {
        const float us = fmaf((float)m - 0.5f * (float)(nu - 1), d.du, off_u);
        row[m] = 0.f;
        row[2 * nu + m] = 0.f;
        row[nu + m] = __ldg(src + m) * (d.sdd / sqrtf(fmaf(d.sdd, d.sdd, fmaf(us, us, vs * vs))));
    }
    __syncthreads();
    for (int n = threadIdx.x; n < nu; n += blockDim.x) {
        const float *c = row + nu + n;
        double acc = (double)scale0 * (double)c[0];        // D h[0] p1[n]
        for (int k = 1; k < nu; k += 2) acc += (double)__ldg(hk + (k >> 1)) * (double)(c[-k] + c[k]);
        q[((size_t)a * d.nv + v) * nu + n] = (float)acc;
    }
}

template <int KC>
__global__ void __launch_bounds__(128)
fdk_backproject_kernel(const DevGeom d, const float *__restrict__ q, const float scale, float *__restrict__ out)
{
    const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * 4 + threadIdx.y, k0 = blockIdx.z * KC;
    if (i >= d.nx || j >= d.ny) return;
    const float x = ((float)i - 0.5f * (float)(d.nx - 1)) * d.hx, y = ((float)j - 0.5f * (float)(d.ny - 1)) * d.hy;
    const float z0 = ((float)k0 - 0.5f * (float)(d.nz - 1)) * d.hz;
    const float inv_du = 1.f / d.du, inv_dv = 1.f / d.dv;
    float acc[KC];
#pragma unroll
    for (int m = 0; m < KC; ++m) acc[m] = 0.f;
    for (int a = 0; a < d.na; ++a) {
        const float2 cs = __ldg(d.cs + a);
        const float U = d.sad - fmaf(x, cs.x, y * cs.y);           // > 0: the volume lies between source and detector
        const float lat = fmaf(-x, cs.y, y * cs.x);
        const float inv_U = 1.f / U, M = d.sdd * inv_U;
        const float pu = fmaf(M * lat, inv_du, d.cu);
        const float fu = floorf(pu), au = pu - fu;
        const int iu = (int)fu;
        const bool u0ok = (unsigned)iu < (unsigned)d.nu, u1ok = (unsigned)(iu + 1) < (unsigned)d.nu;
        if (!u0ok && !u1ok) continue;
        const float w0 = u0ok ? 1.f - au : 0.f, w1 = u1ok ? au : 0.f;
        const float *img = q + (size_t)a * d.nv * d.nu;
        const int c0 = min(max(iu, 0), d.nu - 1), c1 = min(max(iu + 1, 0), d.nu - 1);
        const float wgt = (d.sad * inv_U) * (d.sad * inv_U), Mv = M * inv_dv;
#pragma unroll
        for (int m = 0; m < KC; ++m) {
            const float pv = fmaf(Mv, fmaf((float)m, d.hz, z0), d.cv);
            const float fv = floorf(pv), av = pv - fv;
            const int iv = (int)fv;
            const bool v0ok = (unsigned)iv < (unsigned)d.nv, v1ok = (unsigned)(iv + 1) < (unsigned)d.nv;
            const int row0 = min(max(iv, 0), d.nv - 1) * d.nu, row1 = min(max(iv + 1, 0), d.nv - 1) * d.nu;
            const float b0 = fmaf(w0, __ldg(img + (row0 + c0)), w1 * __ldg(img + (row0 + c1)));
            const float b1 = fmaf(w0, __ldg(img + (row1 + c0)), w1 * __ldg(img + (row1 + c1)));
            acc[m] = fmaf(wgt, fmaf(v0ok ? 1.f - av : 0.f, b0, (v1ok ? av : 0.f) * b1), acc[m]);
        }
    }
#pragma unroll
    for (int m = 0; m < KC; ++m) {
        const int k = k0 + m;
        if (k >= d.nz) break;
        out[((size_t)k * d.ny + j) * d.nx + i] = scale * acc[m];
    }
}
}  // namespace

extern "C" cbct_status cbct_fdk_reconstruct(const cbct_geometry *gc, const float *d_Y, float *d_vol, void *stream)
{
    if (!gc || !d_Y || !d_vol) { cbct_set_error("cbct_fdk_reconstruct: NULL argument"); return CBCT_ERR_INVALID_ARG; }
    cbct_geometry *g = const_cast<cbct_geometry *>(gc);
    cudaStream_t st = (cudaStream_t)stream;
    if ((size_t)3 * g->nu * sizeof(float) > 200 * 1024) {
        cbct_set_error("cbct_fdk_reconstruct: nu = %d exceeds the shared-memory row buffer (nu <= 17066)", g->nu);
        return CBCT_ERR_SHAPE;
    }
    CBCT_TRY(ensure(g, &g->fdk_q, g->n_proj()));
    const double D = g->du * g->sad / g->sdd, kPi = 3.14159265358979323846;
    if (!g->fdk_hk) {                                      // D h[k] for odd k = 1, 3, ... (fp64 on the host, stored fp32)
        std::vector<float> hk((size_t)(g->nu + 1) / 2 + 1);
        for (size_t m = 0; m < hk.size(); ++m) {
            const double k = 2.0 * (double)m + 1.0;
            hk[m] = (float)(-1.0 / (kPi * kPi * k * k * D));
        }
        CBCT_TRY(cbct_dev_alloc(g, (void **)&g->fdk_hk, hk.size() * sizeof(float), false, nullptr));
        CBCT_CUDA(cudaMemcpyAsync(g->fdk_hk, hk.data(), hk.size() * sizeof(float), cudaMemcpyHostToDevice, st));
        CBCT_CUDA(cudaStreamSynchronize(st));              // hk is a host temporary
    }
    {
        ProfileScope ps(1, st);
        const size_t smem = (size_t)3 * g->nu * sizeof(float);
        if (smem > 48 * 1024) CBCT_CUDA(cudaFuncSetAttribute(fdk_filter_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        fdk_filter_kernel<<<dim3(g->nv, g->na), 256, smem, st>>>(g->dev, d_Y, g->fdk_hk, g->fdk_q, (float)g->off_u, (float)g->off_v,
                                                                 (float)(1.0 / (4.0 * D)));
        CBCT_LAUNCH_CHECK();
    }
    {
        constexpr int KC = 8;
        ProfileScope ps(3, st);
        dim3 grid((g->nx + 31) / 32, (g->ny + 3) / 4, (g->nz + KC - 1) / KC), block(32, 4);
        fdk_backproject_kernel<KC><<<grid, block, 0, st>>>(g->dev, g->fdk_q, (float)(kPi / g->na), d_vol);
        CBCT_LAUNCH_CHECK();
    }
    return CBCT_OK;
}
