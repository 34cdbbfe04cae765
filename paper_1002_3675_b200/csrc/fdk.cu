// NEXT-4: the FDK reconstruction the paper compares against (Feldkamp, Davis, Kress = ref. 1; Fig. 1(d) at P:105,
// Fig. 2 at P:125).  Reading Q22 of DESIGN.md: equally spaced views over a full rotation, no redundancy weights, no window.
//   1. p1 = Y SDD / sqrt(SDD^2 + us^2 + vs^2)                                   (cosine pre-weight, fused into the row load)
//   2. q[n] = D sum_m h[n-m] p1[m],  D = du SAD/SDD,  h[0] = 1/(4 D^2), h[even] = 0, h[odd k] = -1/(pi^2 k^2 D^2)
//   3. f(x) = (pi / N_theta) sum_a SAD^2/U^2 q_a(u*, v*),  U = SAD - (x cos a + y sin a), (u*, v*) = SDD (lat, z)/U, bilinear
#include "cbct_internal.h"

namespace {
// One CTA per detector row (a, v).  The pre-weighted row sits in shared memory with nu zeros on either side, so that the
// symmetric pairs p1[n-k] + p1[n+k] need no bounds test; only odd k carry weight.  Direct convolution: nu^2/2 FMAs per row
// (2e9 for 40 views of 512 x 384), no FFT and no library on the path.  Everything up to the stored result is fp64 - the
// pre-weight, the row, the taps and the sum: the ramp filter removes the row's mean, so the result is ~100x smaller than its
// largest terms, and ANY fp32 rounding before the sum (of the weighted row, of a tap, of the centre weight) comes back 100x
// larger relative to q (measured: 7.8e-6 of the oracle on c3's line integrals with an fp32 row and fp32 taps, against 1.4e-7
// on white noise, where nothing cancels).  sm_100 runs fp64 FMAs at half the fp32 rate; the sum was fp64 already.
__global__ void __launch_bounds__(256)
fdk_filter_kernel(const DevGeom d, const float *__restrict__ Y, const double *__restrict__ hk, float *__restrict__ q,
                  const double du, const double dv, const double sdd, const double off_u, const double off_v, const double scale0)
{
    extern __shared__ double row[];                        // [3 nu]: zeros | p1 | zeros
    const int v = blockIdx.x, a = blockIdx.y, nu = d.nu;
    const double vs = fma((double)v - 0.5 * (double)(d.nv - 1), dv, off_v);
    const float *src = Y + ((size_t)a * d.nv + v) * nu;
    for (int m = threadIdx.x; m < nu; m += blockDim.x) {
        const double us = fma((double)m - 0.5 * (double)(nu - 1), du, off_u);
        row[m] = 0.0;
        row[2 * nu + m] = 0.0;
        row[nu + m] = (double)__ldg(src + m) * (sdd / sqrt(fma(sdd, sdd, fma(us, us, vs * vs))));
    }
    __syncthreads();
    for (int n = threadIdx.x; n < nu; n += blockDim.x) {
        const double *c = row + nu + n;
        double acc = scale0 * c[0];                        // D h[0] p1[n]
        for (int k = 1; k < nu; k += 2) acc = fma(__ldg(hk + (k >> 1)), c[-k] + c[k], acc);
        q[((size_t)a * d.nv + v) * nu + n] = (float)acc;
    }
}

// Detector coordinates in fp64.  A voxel's detector column reaches nu/2 pixels from the central ray (256 at c3), where one
// fp32 ulp is 3e-5 pixel, and the ramp-filtered rows change by their own size within a pixel: with (u*, v*) in fp32 (and
// cos, sin rounded to fp32) the full-size c3 volume sat at 1.2e-5 of the oracle.  The u arithmetic is shared by the KC voxels
// of a thread's z column and sm_100 has a full-rate fp64 pipe, so the positions are simply computed in fp64 from the handle's
// fp64 geometry; the fractional weights, the bilinear blend and the sum over the views stay in fp32.
struct FdkGeom {
    double sad, sdd, hx, hy, hz, inv_du, inv_dv, cu, cv;     // cu, cv: detector index of the central ray
};

template <int KC>
__global__ void __launch_bounds__(128)
fdk_backproject_kernel(const DevGeom d, const FdkGeom e, const double2 *__restrict__ cs64, const float *__restrict__ q,
                       const float scale, float *__restrict__ out)
{
    const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * 4 + threadIdx.y, k0 = blockIdx.z * KC;
    if (i >= d.nx || j >= d.ny) return;
    const double x = ((double)i - 0.5 * (double)(d.nx - 1)) * e.hx, y = ((double)j - 0.5 * (double)(d.ny - 1)) * e.hy;
    double z[KC];
    float acc[KC];
#pragma unroll
    for (int m = 0; m < KC; ++m) {
        z[m] = ((double)(k0 + m) - 0.5 * (double)(d.nz - 1)) * e.hz;
        acc[m] = 0.f;
    }
    for (int a = 0; a < d.na; ++a) {
        const double2 cs = __ldg(cs64 + a);
        const double U = e.sad - fma(x, cs.x, y * cs.y);           // > 0: the volume lies between source and detector
        const double lat = fma(-x, cs.y, y * cs.x);
        const double inv_U = 1.0 / U, M = e.sdd * inv_U;
        const double pu = fma(M * lat, e.inv_du, e.cu);
        const double fu = floor(pu);
        const float au = (float)(pu - fu);
        const int iu = (int)fu;
        const bool u0ok = (unsigned)iu < (unsigned)d.nu, u1ok = (unsigned)(iu + 1) < (unsigned)d.nu;
        if (!u0ok && !u1ok) continue;
        const float w0 = u0ok ? 1.f - au : 0.f, w1 = u1ok ? au : 0.f;
        const float *img = q + (size_t)a * d.nv * d.nu;
        const int c0 = min(max(iu, 0), d.nu - 1), c1 = min(max(iu + 1, 0), d.nu - 1);
        const float sU = (float)(e.sad * inv_U), wgt = sU * sU;
        const double Mv = M * e.inv_dv;
#pragma unroll
        for (int m = 0; m < KC; ++m) {
            const double pv = fma(Mv, z[m], e.cv);
            const double fv = floor(pv);
            const float av = (float)(pv - fv);
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

// The weight pi / N_theta per view is the quadrature of a full turn in equal steps (Q22): the list must be
// angles[0] + s * 2 pi a / N, s = +1 or -1, to 1e-6 of a step.
bool equally_spaced_full_turn(const std::vector<double> &ang)
{
    const size_t n = ang.size();
    if (n < 2) return true;
    const double kTwoPi = 6.28318530717958647692, step = kTwoPi / (double)n;
    const double sgn = ang[1] >= ang[0] ? 1.0 : -1.0;
    for (size_t a = 1; a < n; ++a)
        if (!(std::fabs((ang[a] - ang[a - 1]) - sgn * step) <= 1e-6 * step)) return false;
    return true;
}
}  // namespace

extern "C" cbct_status cbct_fdk_reconstruct(const cbct_geometry *gc, const float *d_Y, float *d_vol, void *stream)
{
    if (!gc || !d_Y || !d_vol) { cbct_set_error("cbct_fdk_reconstruct: NULL argument"); return CBCT_ERR_INVALID_ARG; }
    cbct_geometry *g = const_cast<cbct_geometry *>(gc);
    cudaStream_t st = (cudaStream_t)stream;
    if ((size_t)3 * g->nu * sizeof(double) > 200 * 1024) {
        cbct_set_error("cbct_fdk_reconstruct: nu = %d exceeds the shared-memory row buffer (nu <= 8533)", g->nu);
        return CBCT_ERR_SHAPE;
    }
    if (!equally_spaced_full_turn(g->angles)) {
        cbct_set_error("cbct_fdk_reconstruct: the %d views are not equally spaced over a full rotation (the weight pi/N_theta "
                       "per view holds for that scan only; short scans need redundancy weights this routine does not apply)", g->na);
        return CBCT_ERR_SHAPE;
    }
    CBCT_TRY(ensure(g, &g->fdk_q, g->n_proj()));
    const double D = g->du * g->sad / g->sdd, kPi = 3.14159265358979323846;
    if (!g->fdk_hk) {                                      // D h[k] for odd k = 1, 3, ... (fp64)
        std::vector<double> hk((size_t)(g->nu + 1) / 2 + 1);
        for (size_t m = 0; m < hk.size(); ++m) {
            const double k = 2.0 * (double)m + 1.0;
            hk[m] = -1.0 / (kPi * kPi * k * k * D);
        }
        CBCT_TRY(cbct_dev_alloc(g, (void **)&g->fdk_hk, hk.size() * sizeof(double), false, nullptr));
        CBCT_CUDA(cudaMemcpyAsync(g->fdk_hk, hk.data(), hk.size() * sizeof(double), cudaMemcpyHostToDevice, st));
        std::vector<double2> cs((size_t)g->na);            // cos, sin of the views in fp64 (the fp32 table of the march drops 6e-8)
        for (int a = 0; a < g->na; ++a) cs[a] = make_double2(std::cos(g->angles[a]), std::sin(g->angles[a]));
        CBCT_TRY(cbct_dev_alloc(g, (void **)&g->fdk_cs, cs.size() * sizeof(double2), false, nullptr));
        CBCT_CUDA(cudaMemcpyAsync(g->fdk_cs, cs.data(), cs.size() * sizeof(double2), cudaMemcpyHostToDevice, st));
        CBCT_CUDA(cudaStreamSynchronize(st));              // hk and cs are host temporaries
    }
    {
        ProfileScope ps(1, st);
        const size_t smem = (size_t)3 * g->nu * sizeof(double);
        if (smem > 48 * 1024) CBCT_CUDA(cudaFuncSetAttribute(fdk_filter_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        fdk_filter_kernel<<<dim3(g->nv, g->na), 256, smem, st>>>(g->dev, d_Y, g->fdk_hk, g->fdk_q, g->du, g->dv, g->sdd, g->off_u, g->off_v,
                                                                 1.0 / (4.0 * D));
        CBCT_LAUNCH_CHECK();
    }
    {
        constexpr int KC = 8;
        ProfileScope ps(3, st);
        dim3 grid((g->nx + 31) / 32, (g->ny + 3) / 4, (g->nz + KC - 1) / KC), block(32, 4);
        const FdkGeom e = {g->sad, g->sdd, g->hx, g->hy, g->hz, 1.0 / g->du, 1.0 / g->dv,
                           0.5 * (double)(g->nu - 1) - g->off_u / g->du, 0.5 * (double)(g->nv - 1) - g->off_v / g->dv};
        fdk_backproject_kernel<KC><<<grid, block, 0, st>>>(g->dev, e, g->fdk_cs, g->fdk_q, (float)(kPi / g->na), d_vol);
        CBCT_LAUNCH_CHECK();
    }
    return CBCT_OK;
}
