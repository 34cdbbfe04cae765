// Geometry handle: validation, fp64 ray tables, coarse levels, scratch bookkeeping.
// Convention O0 of DESIGN.md (the paper fixes none of it).
#include <cmath>
#include <cstdarg>
#include <cstring>
#include <new>

#include "cbct_internal.h"

std::atomic<unsigned long long> g_cbct_launches{0};
static thread_local char t_err[512] = "";

void cbct_set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof(t_err), fmt, ap);
    va_end(ap);
}

extern "C" const char *cbct_last_error(void) { return t_err; }
extern "C" unsigned long long cbct_launch_count(void) { return g_cbct_launches.load(); }

// Guard mode (cbct_set_guard_mode): every device buffer a handle allocates from then on sits between two kGuard-byte
// regions filled with a pattern; cbct_check_guards counts the pattern bytes that changed.  It stands in for compute-sanitizer's
// memcheck, which this pool does not allow: an out-of-bounds WRITE of any kernel into library-owned memory shows up there.
static constexpr size_t kGuard = 4096;
static constexpr unsigned char kGuardByte = 0xA5;
static std::atomic<int> g_guard_mode{0};

extern "C" cbct_status cbct_set_guard_mode(int on)
{
    g_guard_mode.store(on != 0);
    return CBCT_OK;
}

cbct_status cbct_dev_alloc(cbct_geometry *g, void **p, size_t bytes, bool zero, cudaStream_t st)
{
    const bool guard = g_guard_mode.load() != 0;
    const size_t padded = (bytes + 255) / 256 * 256;            // the rear guard starts on a 256-byte boundary behind the buffer
    void *base = nullptr;
    cudaError_t e = cudaMalloc(&base, guard ? padded + 2 * kGuard : bytes);
    if (e != cudaSuccess) {
        *p = nullptr;
        cudaGetLastError();
        cbct_set_error("cudaMalloc(%zu bytes) failed: %s", bytes, cudaGetErrorString(e));
        return CBCT_ERR_ALLOC;
    }
    if (guard) {
        // whole allocation patterned (so the slack up to `padded` is guarded too), then waited for: debug mode
        CBCT_CUDA(cudaMemset(base, kGuardByte, padded + 2 * kGuard));
        CBCT_CUDA(cudaDeviceSynchronize());
        *p = static_cast<char *>(base) + kGuard;
        g->guarded.push_back({*p, bytes, padded});
    } else {
        *p = base;
    }
    // zero-fill ON THE CALLER'S STREAM: the first kernel that touches the buffer is launched on it right afterwards,
    // and nothing orders the legacy default stream against a non-blocking stream (PyTorch's side streams)
    if (zero) CBCT_CUDA(cudaMemsetAsync(*p, 0, bytes, st));
    g->bytes += bytes;
    return CBCT_OK;
}

void cbct_dev_free(cbct_geometry *g, void *p)
{
    if (!p) return;
    for (size_t n = 0; n < g->guarded.size(); ++n)
        if (g->guarded[n].ptr == p) {
            cudaFree(static_cast<char *>(p) - kGuard);
            g->guarded.erase(g->guarded.begin() + n);
            return;
        }
    cudaFree(p);
}

extern "C" cbct_status cbct_check_guards(const cbct_geometry *gc, unsigned long long *h_bad_bytes)
{
    if (!gc || !h_bad_bytes) { cbct_set_error("cbct_check_guards: NULL argument"); return CBCT_ERR_INVALID_ARG; }
    *h_bad_bytes = 0;
    CBCT_CUDA(cudaDeviceSynchronize());
    std::vector<unsigned char> h;
    for (const cbct_geometry *g = gc; g; g = g->coarse)
        for (const auto &b : g->guarded) {
            const char *user = static_cast<const char *>(b.ptr);
            // front guard, then everything from the end of the user's bytes to the end of the rear guard
            const struct { const char *at; size_t n; } spans[2] = {{user - kGuard, kGuard}, {user + b.bytes, b.padded - b.bytes + kGuard}};
            for (const auto &sp : spans) {
                h.resize(sp.n);
                CBCT_CUDA(cudaMemcpy(h.data(), sp.at, sp.n, cudaMemcpyDeviceToHost));
                for (unsigned char c : h) *h_bad_bytes += c != kGuardByte;
            }
        }
    return CBCT_OK;
}

static void free_handle(cbct_geometry *g)
{
    if (!g) return;
    free_handle(g->coarse);
    void *ptrs[] = {g->d_rays, g->d_rays_lo, g->d_zeta, g->d_inv_zeta, g->d_dz, g->d_cs, g->d_tiles[0], g->d_tiles[1],
                    g->d_angle_has[0], g->d_angle_has[1], g->vol_pad[0], g->vol_pad[1], g->proj_tmp, g->proj_prefix,
                    g->G_cls[0], g->G_cls[1], g->vol_a, g->vol_b, g->vol_c, g->vol_f, g->Y_level, g->vc_tau, g->vc_f0, g->vc_d, g->vc_e, g->fdk_q, g->fdk_hk, g->fdk_cs,
                    g->red_partial, g->red_out, g->host_stage_vol, g->host_stage_proj, g->host_stage_vol2};
    for (void *p : ptrs) cbct_dev_free(g, p);
    if (g->h_red) cudaFreeHost(g->h_red);
    if (g->graph_stream) cudaStreamDestroy(g->graph_stream);
    if (g->copy_stream) cudaStreamDestroy(g->copy_stream);
    if (g->ev_f0) cudaEventDestroy(g->ev_f0);
    if (g->ev_Y) cudaEventDestroy(g->ev_Y);
    delete g;
}

extern "C" void cbct_geometry_destroy(cbct_geometry *g)
{
    if (!g) return;
    cudaDeviceSynchronize();
    free_handle(g);
}

extern "C" unsigned long long cbct_device_bytes(const cbct_geometry *g)
{
    unsigned long long b = 0;
    for (const cbct_geometry *q = g; q; q = q->coarse) b += q->bytes;
    return b;
}

extern "C" cbct_status cbct_geometry_query(const cbct_geometry *g, int *d6, double *s5)
{
    if (!g) { cbct_set_error("cbct_geometry_query: NULL handle"); return CBCT_ERR_INVALID_ARG; }
    if (d6) { d6[0] = g->na; d6[1] = g->nu; d6[2] = g->nv; d6[3] = g->nx; d6[4] = g->ny; d6[5] = g->nz; }
    if (s5) { s5[0] = g->du; s5[1] = g->dv; s5[2] = g->hx; s5[3] = g->hy; s5[4] = g->hz; }
    return CBCT_OK;
}

template <typename T>
static cbct_status upload(cbct_geometry *g, T **dst, const std::vector<T> &src)
{
    if (src.empty()) { *dst = nullptr; return CBCT_OK; }
    CBCT_TRY(cbct_dev_alloc(g, (void **)dst, src.size() * sizeof(T), false, nullptr));
    CBCT_CUDA(cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice));
    return CBCT_OK;
}

static cbct_status build_tables(cbct_geometry *g)
{
    const int na = g->na, nu = g->nu, nv = g->nv;
    DevGeom &d = g->dev;
    d.na = na; d.nu = nu; d.nv = nv; d.nx = g->nx; d.ny = g->ny; d.nz = g->nz;
    d.koff = g->nz / 2;
    d.zfrac = (float)(0.5 * g->nz - d.koff);
    d.hx = (float)g->hx; d.hy = (float)g->hy; d.hz = (float)g->hz;
    d.du = (float)g->du; d.dv = (float)g->dv; d.sad = (float)g->sad; d.sdd = (float)g->sdd;
    d.cu = (float)(0.5 * (nu - 1) - g->off_u / g->du);
    d.cv = (float)(0.5 * (nv - 1) - g->off_v / g->dv);
    d.cv_lo = (float)((0.5 * (nv - 1) - g->off_v / g->dv) - (double)d.cv);
    d.hzdv_hi = (float)(g->hz / g->dv);
    d.hzdv_lo = (float)(g->hz / g->dv - (double)d.hzdv_hi);
    for (int c = 0; c < 2; ++c) {
        ClassGrid &cg = d.cls[c];
        cg.nmaj = c == 0 ? g->nx : g->ny;
        cg.nmin = c == 0 ? g->ny : g->nx;
        cg.hmaj = (float)(c == 0 ? g->hx : g->hy);
        cg.hmin = (float)(c == 0 ? g->hy : g->hx);
        cg.ioff = cg.nmaj / 2;
        cg.joff = cg.nmin / 2;
        cg.row_stride = ((cg.nmin + kPadLo + kPadHi + 3) / 4) * 4;
        cg.plane_stride = (long long)cg.nmaj * cg.row_stride;
        if ((long long)(g->nz + 2 * kPadK) * cg.plane_stride >= (1LL << 31)) {
            cbct_set_error("geometry unsupported: the padded volume copy has 2^31 or more elements (32-bit offsets in the march)");
            return CBCT_ERR_SHAPE;
        }
    }

    std::vector<RayXY> rays((size_t)na * nu);
    std::vector<float4> rays_lo((size_t)na * nu);
    std::vector<float2> cs(na);
    std::vector<float> zeta(nv), inv_zeta(nv), dz(nv);
    double max_abs_zeta = 0.0;
    for (int v = 0; v < nv; ++v) {
        double Dz = (v - 0.5 * (nv - 1)) * g->dv + g->off_v;
        dz[v] = (float)Dz;
        // A ray with Dz == 0 (centre row of an odd nv) never leaves its z row.  It is given an
        // infinitesimal positive slope so that sign(sz) and sign(1/sz) agree in the kernels and a
        // ray lying exactly in a z plane is assigned to the row above it, as floor() would.
        zeta[v] = Dz != 0.0 ? (float)(Dz / g->hz) : 1e-30f;
        inv_zeta[v] = Dz != 0.0 ? (float)(g->hz / Dz) : 1e30f;
        max_abs_zeta = std::fmax(max_abs_zeta, std::fabs(Dz / g->hz));
    }
    std::vector<int2> tiles[2];
    double max_abs_dt = 0.0, t_min = 1.0;
    for (int c = 0; c < 2; ++c) g->h_angle_has[c].assign(na, 0);
    for (int a = 0; a < na; ++a) {
        const double th = g->angles[a], co = std::cos(th), si = std::sin(th);
        cs[a] = make_float2((float)co, (float)si);
        const double Sx = g->sad * co, Sy = g->sad * si;
        for (int u = 0; u < nu; ++u) {
            const double uc = (u - 0.5 * (nu - 1)) * g->du + g->off_u;
            const double Dx = -(g->sdd - g->sad) * co - uc * si;
            const double Dy = -(g->sdd - g->sad) * si + uc * co;
            const double dXv = (Dx - Sx) / g->hx, dYv = (Dy - Sy) / g->hy;
            const int c = std::fabs(dXv) >= std::fabs(dYv) ? 0 : 1;
            const ClassGrid &cg = d.cls[c];
            const double Smaj = c == 0 ? Sx : Sy, Smin = c == 0 ? Sy : Sx;
            const double dmaj = c == 0 ? Dx - Sx : Dy - Sy, dmin = c == 0 ? Dy - Sy : Dx - Sx;
            const double hmaj = c == 0 ? g->hx : g->hy;
            const double hmin = c == 0 ? g->hy : g->hx;
            const double sm = (dmin / hmin) / (dmaj / hmaj);
            const double dt = hmaj / dmaj;
            const double tc = ((cg.ioff - 0.5 * cg.nmaj) * hmaj - Smaj) / dmaj;
            const double mcu = (Smin + tc * dmin) / hmin + 0.5 * cg.nmin;   // un-centred minor coordinate at plane ioff
            RayXY r;
            r.mc = (float)(mcu - cg.joff);
            r.sm = (float)sm;
            r.inv_sm = sm != 0.0 ? (float)(1.0 / sm) : 1e30f;
            if ((float)sm == 0.f) r.inv_sm = 1e30f;
            r.tc = (float)tc;
            r.dt = (float)dt;
            r.inv_dt = (float)(1.0 / dt);
            r.lxy2 = (float)(hmaj * hmaj + sm * hmin * sm * hmin);
            // slabs i (between major planes i and i+1) where the minor coordinate can lie in [-1, nmin+1]
            int ilo = 0, ihi = cg.nmaj;
            if (sm != 0.0) {
                double e0 = (-1.0 - mcu) / sm, e1 = (cg.nmin + 1.0 - mcu) / sm;
                double lo = std::fmin(e0, e1) + cg.ioff, hi = std::fmax(e0, e1) + cg.ioff;
                double flo = std::floor(lo) - 1.0, fhi = std::ceil(hi) + 1.0;
                if (flo > ilo) ilo = flo > cg.nmaj ? cg.nmaj : (int)flo;
                if (fhi < ihi) ihi = fhi < 0 ? 0 : (int)fhi;
            } else if (mcu < -1.0 || mcu > cg.nmin + 1.0) {
                ihi = 0;
            }
            if (ihi < ilo) ihi = ilo;
            r.range = ilo | (ihi << 15) | (c << 30);
            rays[(size_t)a * nu + u] = r;
            rays_lo[(size_t)a * nu + u] = make_float4((float)((mcu - cg.joff) - (double)r.mc), (float)(sm - (double)r.sm),
                                                      (float)(tc - (double)r.tc), 0.f);
            if (ihi > ilo) {
                g->h_angle_has[c][a] = 1;
                max_abs_dt = std::fmax(max_abs_dt, std::fabs(dt));
                t_min = std::fmin(t_min, std::fmin(tc + (ilo - cg.ioff) * dt, tc + (ihi - cg.ioff) * dt));
            }
        }
        for (int c = 0; c < 2; ++c)
            for (int u0 = 0; u0 < nu; u0 += 32) {
                // every ray is written by exactly one launch (the one of its class), whether it meets the volume or
                // not: a tile is listed for class c as soon as it holds a ray of class c, so rays that miss still get
                // their 0 (mode 0) or -Y (residual modes) and nothing stale survives in the output
                bool any = false;
                for (int u = u0; u < u0 + 32 && u < nu; ++u)
                    if (ray_cls(rays[(size_t)a * nu + u].range) == c) any = true;
                if (any) tiles[c].push_back(make_int2(a, u0));
            }
    }
    g->max_abs_sz = (float)(max_abs_dt * max_abs_zeta);
    g->bp_run_max = (float)(std::ceil((g->hz / g->dv) / std::fmax(t_min, 1e-3)) + 2.0);
    if (g->max_abs_sz > 0.999f) {
        cbct_set_error("geometry unsupported: a ray climbs %.3f voxels in z per major-axis voxel (limit 0.999)",
                       g->max_abs_sz);
        return CBCT_ERR_SHAPE;
    }
    CBCT_TRY(upload(g, &g->d_rays, rays));
    CBCT_TRY(upload(g, &g->d_rays_lo, rays_lo));
    CBCT_TRY(upload(g, &g->d_cs, cs));
    CBCT_TRY(upload(g, &g->d_zeta, zeta));
    CBCT_TRY(upload(g, &g->d_inv_zeta, inv_zeta));
    CBCT_TRY(upload(g, &g->d_dz, dz));
    // the angle list closed under + 180 degrees, second half in the order of the first?
    g->twin_ok = na % 2 == 0 && na >= 2;
    for (int a = 0; g->twin_ok && a < na / 2; ++a) {
        const double dlt = std::remainder(g->angles[a + na / 2] - g->angles[a] - 3.14159265358979323846, 2.0 * 3.14159265358979323846);
        if (std::fabs(dlt) > 1e-12) g->twin_ok = false;
    }
    for (int c = 0; c < 2; ++c) {
        g->n_tiles[c] = (int)tiles[c].size();
        g->n_tiles_half[c] = 0;
        for (const int2 &t : tiles[c]) g->n_tiles_half[c] += t.x < na / 2;
        CBCT_TRY(upload(g, &g->d_tiles[c], tiles[c]));
        CBCT_TRY(upload(g, &g->d_angle_has[c], g->h_angle_has[c]));
    }
    d.rays = g->d_rays; d.rays_lo = g->d_rays_lo; d.cs = g->d_cs; d.zeta = g->d_zeta; d.inv_zeta = g->d_inv_zeta; d.dz_mm = g->d_dz;
    // the table uploads are cudaMemcpy's from pageable memory on the legacy default stream: wait for them here, so that the
    // first kernel may run on any (also a non-blocking) stream
    CBCT_CUDA(cudaStreamSynchronize(nullptr));
    return CBCT_OK;
}

static cbct_status create_impl(double sad, double sdd, const double *angles, int na, int nu, int nv,
                               double du, double dv, int nx, int ny, int nz, double hx, double hy, double hz,
                               double off_u, double off_v, cbct_geometry **out)
{
    if (!out) { cbct_set_error("cbct_geometry_create: out is NULL"); return CBCT_ERR_INVALID_ARG; }
    *out = nullptr;
    if (!angles || na <= 0 || nu <= 0 || nv <= 0 || nx <= 0 || ny <= 0 || nz <= 0 ||
        !(du > 0) || !(dv > 0) || !(hx > 0) || !(hy > 0) || !(hz > 0) || !(sad > 0) || !(sdd > sad) ||
        !std::isfinite(off_u) || !std::isfinite(off_v)) {
        cbct_set_error("cbct_geometry_create: NULL angles, non-positive size, sad >= sdd, or a non-finite detector offset");
        return CBCT_ERR_INVALID_ARG;
    }
    for (int a = 0; a < na; ++a)
        if (!std::isfinite(angles[a])) { cbct_set_error("cbct_geometry_create: non-finite angle"); return CBCT_ERR_INVALID_ARG; }
    if (nx > 16384 || ny > 16384 || nz > 16384 || nu > 16384 || nv > 16384) {
        cbct_set_error("cbct_geometry_create: a dimension exceeds 16384");
        return CBCT_ERR_SHAPE;
    }
    if ((long long)na * (nv + 1) * nu >= (1LL << 31)) {
        cbct_set_error("cbct_geometry_create: n_angles * (nv + 1) * nu must stay below 2^31 (32-bit offsets in the gather)");
        return CBCT_ERR_SHAPE;
    }
    const double rad = 0.5 * std::hypot(nx * hx, ny * hy);
    if (!(rad < sad) || !(rad < sdd - sad)) {
        cbct_set_error("cbct_geometry_create: the volume's circumscribed cylinder (r=%.1f mm) is not strictly "
                       "between source (%.1f) and detector (%.1f)", rad, sad, sdd - sad);
        return CBCT_ERR_SHAPE;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        cbct_set_error("no CUDA device (libcbct has no CPU fallback)");
        return CBCT_ERR_CUDA;
    }
    cbct_geometry *g = new (std::nothrow) cbct_geometry();
    if (!g) { cbct_set_error("out of host memory"); return CBCT_ERR_ALLOC; }
    g->sad = sad; g->sdd = sdd; g->du = du; g->dv = dv; g->hx = hx; g->hy = hy; g->hz = hz;
    g->off_u = off_u; g->off_v = off_v;
    g->na = na; g->nu = nu; g->nv = nv; g->nx = nx; g->ny = ny; g->nz = nz;
    g->angles.assign(angles, angles + na);
    cbct_status s = build_tables(g);
    if (s != CBCT_OK) { free_handle(g); return s; }
    *out = g;
    return CBCT_OK;
}

extern "C" cbct_status cbct_geometry_create(double sad, double sdd, const double *angles, int na, int nu, int nv,
                                            double du, double dv, int nx, int ny, int nz,
                                            double hx, double hy, double hz, cbct_geometry **out)
{
    return create_impl(sad, sdd, angles, na, nu, nv, du, dv, nx, ny, nz, hx, hy, hz, 0.0, 0.0, out);
}

extern "C" cbct_status cbct_geometry_create_ex(double sad, double sdd, const double *angles, int na, int nu, int nv,
                                               double du, double dv, double off_u, double off_v, int nx, int ny, int nz,
                                               double hx, double hy, double hz, cbct_geometry **out)
{
    return create_impl(sad, sdd, angles, na, nu, nv, du, dv, nx, ny, nz, hx, hy, hz, off_u, off_v, out);
}

extern "C" cbct_status cbct_set_detector_binning(cbct_geometry *g, int on)
{
    if (!g) { cbct_set_error("cbct_set_detector_binning: NULL handle"); return CBCT_ERR_INVALID_ARG; }
    if ((on != 0) == (g->bin_detector != 0)) return CBCT_OK;
    // the coarse levels were built for the other choice: drop them (they are rebuilt on demand)
    if (g->coarse) {
        CBCT_CUDA(cudaDeviceSynchronize());
        free_handle(g->coarse);
        g->coarse = nullptr;
    }
    g->bin_detector = on != 0;
    return CBCT_OK;
}

// O6 coarsening rule (Q11): axes with spacing <= sqrt(2) * min spacing halve; detector bins iff x and y did.
extern "C" cbct_status cbct_geometry_coarsen(const cbct_geometry *gc, cbct_geometry **out, int *flags4)
{
    cbct_geometry *g = const_cast<cbct_geometry *>(gc);
    if (!g || !out) { cbct_set_error("cbct_geometry_coarsen: NULL argument"); return CBCT_ERR_INVALID_ARG; }
    if (!g->coarse) {
        const double h[3] = {g->hx, g->hy, g->hz};
        int n[3] = {g->nx, g->ny, g->nz};
        double hn[3] = {g->hx, g->hy, g->hz};
        const double m = std::fmin(h[0], std::fmin(h[1], h[2]));
        int fl[4] = {0, 0, 0, 0};
        for (int a = 0; a < 3; ++a) {
            if (h[a] <= std::sqrt(2.0) * m * (1.0 + 1e-9)) {
                if (n[a] % 2) {
                    cbct_set_error("cbct_geometry_coarsen: odd dimension %d on an axis that must coarsen", n[a]);
                    return CBCT_ERR_SHAPE;
                }
                fl[a] = 1; n[a] /= 2; hn[a] *= 2.0;
            }
        }
        int nu = g->nu, nv = g->nv;
        double du = g->du, dv = g->dv;
        if (fl[0] && fl[1] && g->bin_detector) {
            if (nu % 2 || nv % 2) {
                cbct_set_error("cbct_geometry_coarsen: odd detector dimension on a level that bins the detector");
                return CBCT_ERR_SHAPE;
            }
            fl[3] = 1; nu /= 2; nv /= 2; du *= 2.0; dv *= 2.0;
        }
        cbct_geometry *c = nullptr;
        // the mean position of a binned pixel pair is the binned pixel's centre with the SAME panel shift
        CBCT_TRY(create_impl(g->sad, g->sdd, g->angles.data(), g->na, nu, nv, du, dv, n[0], n[1], n[2],
                             hn[0], hn[1], hn[2], g->off_u, g->off_v, &c));
        c->bp_mode = g->bp_mode;
        c->bin_detector = g->bin_detector;
        c->fw_staged = g->fw_staged;
        c->use_mirror = g->use_mirror;
        g->coarse = c;
        std::memcpy(g->coarsen_flags, fl, sizeof(fl));
    }
    *out = g->coarse;
    if (flags4) std::memcpy(flags4, g->coarsen_flags, sizeof(g->coarsen_flags));
    return CBCT_OK;
}
