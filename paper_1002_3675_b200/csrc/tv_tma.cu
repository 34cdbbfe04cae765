// a5/a6, TMA path: the TV-prox Jacobi step (P:89 step 2; O4 in DESIGN.md) for volumes with nx <= 512, nx % 4 == 0.
//
// Same arithmetic as tv_rows.cu, expression by expression:
//   u' = u - dt [ beta (u - g) + grad TV_eps(u) ],  grad TV_eps(u)[ijk] = -(qx+qy+qz)|ijk + qx|i-1 + qy|j-1 + qz|k-1,
//   q_a = (d_a / h_a) / n,  d_a forward difference / h_a (0 at the far face),  n = sqrt(dx^2+dy^2+dz^2+eps^2).
// What changed is how the data move.  A CTA of W warps owns W+1 consecutive rows y0-1 .. y0+W-1 of a chunk of z planes.
// Whole plane tiles of u (W+1 rows, full x extent) are brought into a ring of 4 shared-memory stages by the TMA unit
// (cp.async.bulk.tensor, one elected thread, completion on an mbarrier), two planes ahead of their use: no thread spends
// registers or issue slots on these loads, their addresses or their latency, and rows outside the volume arrive as zeros
// without a bounds test.  g, read once per voxel by the warp that updates it, comes by 16-byte global loads requested before
// the fluxes of the plane (measured on B200, 512^3: g through TMA as well 6.0 TB/s, g by global loads 6.5 TB/s, because the
// smaller stages let the ring run with 8 rows per CTA; a 3-stage ring, one plane ahead, drops to 4.2 TB/s).  A warp owns one x row; lane l holds the float4 chunks at x = 128 q + 4 l, so every
// shared-memory access of a warp is one contiguous 512-byte row segment (conflict-free on the dense TMA layout) and every
// store one 512-byte line group.  Per plane: fluxes of rows y0-1 .. y0+W-2 (qy to the row above through shared memory, one
// barrier), then the update of rows y0 .. y0+W-2 with 16-byte stores.  HBM traffic per voxel and step: read u, read g,
// write u' (12 B), each once (the halo rows of neighbouring CTAs come from L2).
#include <mutex>

#include "cbct_internal.h"
#include "tma.cuh"

namespace {
#ifndef CBCT_TV_STAGES
#define CBCT_TV_STAGES 4
#endif
constexpr int kTvStages = CBCT_TV_STAGES;
#ifndef CBCT_TV_G_LDG
#define CBCT_TV_G_LDG 1
#endif
constexpr bool kGLdg = CBCT_TV_G_LDG != 0;     // g by 16-byte global loads into registers (requested before the fluxes) instead of TMA

// 1/sqrt(x) for normal positive x (x >= eps^2 > 0) in one MUFU instruction
__device__ __forceinline__ float rsqrt_ftz(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <int CH, int W>
struct TvTmaLayout {
    static constexpr int NB = CH > 2 ? 2 : 1;                 // TMA boxes along x (a box is at most 256 elements wide)
    __host__ __device__ static int bx(int nx) { return NB == 2 ? 256 : nx; }
    __host__ __device__ static size_t align128(size_t b) { return (b + 127) & ~(size_t)127; }
    __host__ __device__ static size_t u_bytes(int nx) { return align128((size_t)NB * (W + 1) * bx(nx) * sizeof(float)); }
    __host__ __device__ static size_t g_bytes(int nx) { return kGLdg ? 0 : align128((size_t)NB * (W - 1) * bx(nx) * sizeof(float)); }
    __host__ __device__ static size_t q_bytes(int nx) { return align128((size_t)2 * W * 128 * CH * sizeof(float)); }
    __host__ __device__ static size_t total(int nx) { return kTvStages * (u_bytes(nx) + g_bytes(nx)) + q_bytes(nx) + 128; }
};

template <int CH, int W>
__global__ void __launch_bounds__(32 * W)
tv_tma_kernel(const __grid_constant__ CUtensorMap tm_u, const __grid_constant__ CUtensorMap tm_g, const float *__restrict__ gv,
              float *__restrict__ u_out,
              const int nx, const int ny, const int nz, const float ihx2, const float ihy2, const float ihz2, const float beta,
              const float eps2, const float dt, const float lo_clamp, const int zchunk)
{
    using L = TvTmaLayout<CH, W>;
    constexpr int NB = L::NB, S = kTvStages;
    extern __shared__ __align__(1024) unsigned char smem[];                    // no static shared memory: the window starts aligned
    const int BX = L::bx(nx);
    const size_t ub = L::u_bytes(nx), gb = L::g_bytes(nx);
    float *Ust = reinterpret_cast<float *>(smem);                               // [S][NB][W+1][BX]
    float *Gst = reinterpret_cast<float *>(smem + S * ub);                      // [S][NB][W-1][BX]
    float *Q = reinterpret_cast<float *>(smem + S * (ub + gb));                 // [2][W][128 CH]
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + S * (ub + gb) + L::q_bytes(nx));

    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int y0 = blockIdx.x * (W - 1);
    const int y = y0 - 1 + w;
    const int zc0 = blockIdx.y * zchunk, zc1 = min(zc0 + zchunk, nz);
    const int zs = max(zc0 - 1, 0), zlast = min(zc1, nz - 1);                   // planes zs .. zlast are read
    const bool row_ok = y >= 0 && y < ny;
    const bool do_upd = row_ok && w >= 1;
    const bool has_yp = y + 1 < ny;
    const uint32_t u_tx = (uint32_t)((size_t)NB * (W + 1) * BX * sizeof(float));
    const uint32_t g_tx = (uint32_t)((size_t)NB * (W - 1) * BX * sizeof(float));

    auto issue = [&](int p) {                                                   // one thread: bring plane p into its stage
        const int st = (p - zs) % S;
        const bool with_g = !kGLdg && p >= zc0 && p < zc1;
        mbar_arrive_expect_tx(full + st, u_tx + (with_g ? g_tx : 0u));
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            tma_load_3d(reinterpret_cast<unsigned char *>(Ust) + st * ub + (size_t)b * (W + 1) * BX * sizeof(float), &tm_u, full + st,
                        256 * b, y0 - 1, p);
            if (with_g)
                tma_load_3d(reinterpret_cast<unsigned char *>(Gst) + st * gb + (size_t)b * (W - 1) * BX * sizeof(float), &tm_g,
                            full + st, 256 * b, y0, p);
        }
    };
    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < S; ++s) mbar_init(full + s, 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (threadIdx.x == 0)
        for (int p = zs; p <= zlast && p < zs + S; ++p) issue(p);

    // This lane's float4 chunks sit at x = 128 q + 4 lane: chunk q of a tile row is the float4 at index 32 q + lane of the row
    // (box 0) or of the row's second box (q >= 2 when the row is split into two 256-wide boxes), a compile-time offset from
    // the lane's pointer into the row.  A lane beyond nx (rows shorter than 128 CH) computes on harmless in-bounds data and
    // stores nothing.
    const int row4 = BX / 4;                                                    // float4 per tile row of one box
    auto chunk_off = [&](int q, int rows) { return (NB == 2 && q >= 2) ? rows * row4 + 32 * (q - 2) : 32 * q; };
    bool act[CH];
#pragma unroll
    for (int q = 0; q < CH; ++q) act[q] = 128 * q + 4 * lane < nx;
    const int lane4 = min(lane, row4 - 1);                                      // keeps an idle lane's loads inside the row
    const float4 *U4 = reinterpret_cast<const float4 *>(Ust) + lane4;
    const float4 *G4 = reinterpret_cast<const float4 *>(Gst) + lane4;
    const int ust4 = (int)(ub / 16), gst4 = (int)(gb / 16);                     // float4 per stage
    // rows outside the volume hold zeros (TMA fill); a row that must not produce fluxes (y = -1 or y >= ny) and the far
    // faces (no row above / no plane above) difference the row with itself, which gives exactly zero fluxes
    const int r_own = w * row4, r_up = (row_ok && has_yp ? w + 1 : w) * row4;

    float4 qzp[CH];
#pragma unroll
    for (int q = 0; q < CH; ++q) qzp[q] = make_float4(0.f, 0.f, 0.f, 0.f);

    for (int z = zs; z < zc1; ++z) {
        const int pc = z - zs, stc = pc % S, stn = (pc + 1) % S;
        const bool has_zp = z + 1 < nz;
        mbar_wait(full + stc, (uint32_t)(pc / S) & 1u);
        if (has_zp) mbar_wait(full + stn, (uint32_t)((pc + 1) / S) & 1u);
        float4 *Qc = reinterpret_cast<float4 *>(Q) + (z & 1) * (W * 32 * CH) + lane;       // [W][CH][32] float4
        const float4 *pc4 = U4 + stc * ust4 + r_own, *py4 = U4 + stc * ust4 + r_up;
        const float4 *pn4 = has_zp && row_ok ? U4 + stn * ust4 + r_own : pc4;

        float4 uc[CH], sg[CH];                                                  // u(z) of this row; -(qx+qy+qz) + qx|i-1 + qz|k-1
        float4 gr[kGLdg ? CH : 1];
        const bool upd = do_upd && z >= zc0;
        if (kGLdg && upd) {
            const float4 *gsrc = reinterpret_cast<const float4 *>(gv + ((size_t)z * ny + y) * nx) + lane;
#pragma unroll
            for (int q = 0; q < CH; ++q)
                if (act[q]) gr[kGLdg ? q : 0] = __ldg(gsrc + 32 * q);
        }
#pragma unroll
        for (int q = 0; q < CH; ++q) uc[q] = pc4[chunk_off(q, W + 1)];
        float prev_qx3 = 0.f;                                                   // qx of the last voxel of the previous chunk (this lane)
#pragma unroll
        for (int q = 0; q < CH; ++q) {
            // first voxel of the chunk to the right: lane + 1 of this chunk, or lane 0 of the next chunk
            float xr = __shfl_down_sync(0xffffffffu, uc[q].x, 1);
            if (q + 1 < CH) {
                const float wrap = __shfl_sync(0xffffffffu, uc[q + 1 < CH ? q + 1 : q].x, 0);
                if (lane == 31) xr = wrap;
            }
            const float4 un = pn4[chunk_off(q, W + 1)], uy = py4[chunk_off(q, W + 1)];
            if (128 * q + 4 * lane + 4 >= nx) xr = uc[q].w;                     // no voxel to the right of this chunk
            const float c[4] = {uc[q].x, uc[q].y, uc[q].z, uc[q].w};
            const float r[4] = {uc[q].y, uc[q].z, uc[q].w, xr};
            const float yv[4] = {uy.x, uy.y, uy.z, uy.w}, zv[4] = {un.x, un.y, un.z, un.w};
            float ox[4], oy[4], oz[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const float dx = r[e] - c[e], dy = yv[e] - c[e], dz = zv[e] - c[e];
                const float ex = dx * ihx2, ey = dy * ihy2, ez = dz * ihz2;           // d_a / h_a^2
                const float inv = rsqrt_ftz(fmaf(dx, ex, fmaf(dy, ey, fmaf(dz, ez, eps2))));
                ox[e] = ex * inv; oy[e] = ey * inv; oz[e] = ez * inv;
            }
            Qc[(w * CH + q) * 32] = make_float4(oy[0], oy[1], oy[2], oy[3]);
            // qx of the voxel to the left of the chunk: lane - 1 of this chunk, or lane 31 of the previous chunk (0 at x = 0)
            float qxl = __shfl_up_sync(0xffffffffu, ox[3], 1);
            if (q > 0) {
                const float wrapl = __shfl_sync(0xffffffffu, prev_qx3, 31);
                if (lane == 0) qxl = wrapl;
            } else if (lane == 0) {
                qxl = 0.f;
            }
            prev_qx3 = ox[3];
            sg[q].x = -(ox[0] + oy[0] + oz[0]) + qxl + qzp[q].x;
            sg[q].y = -(ox[1] + oy[1] + oz[1]) + ox[0] + qzp[q].y;
            sg[q].z = -(ox[2] + oy[2] + oz[2]) + ox[1] + qzp[q].z;
            sg[q].w = -(ox[3] + oy[3] + oz[3]) + ox[2] + qzp[q].w;
            qzp[q] = make_float4(oz[0], oz[1], oz[2], oz[3]);
        }
        __syncthreads();
        // every warp is past its reads of plane z-1 (u before the barrier of the previous plane, g after it): refill that stage
        if (threadIdx.x == 0 && z > zs && z - 1 + S <= zlast) issue(z - 1 + S);

        if (upd) {                                                              // warp-uniform
            float4 *dst = reinterpret_cast<float4 *>(u_out + ((size_t)z * ny + y) * nx) + lane;
            const float4 *pg4 = G4 + stc * gst4 + (w - 1) * row4;
#pragma unroll
            for (int q = 0; q < CH; ++q) {
                const float4 qym = Qc[((w - 1) * CH + q) * 32];
                const float4 g = kGLdg ? gr[kGLdg ? q : 0] : pg4[chunk_off(q, W - 1)];
                float4 o;
                // grad = -(qx+qy+qz) + qx|i-1 + qy|j-1 + qz|k-1, summed in the order of tv_rows.cu
                o.x = fmaxf(uc[q].x - dt * fmaf(beta, uc[q].x - g.x, sg[q].x + qym.x), lo_clamp);
                o.y = fmaxf(uc[q].y - dt * fmaf(beta, uc[q].y - g.y, sg[q].y + qym.y), lo_clamp);
                o.z = fmaxf(uc[q].z - dt * fmaf(beta, uc[q].z - g.z, sg[q].z + qym.z), lo_clamp);
                o.w = fmaxf(uc[q].w - dt * fmaf(beta, uc[q].w - g.w, sg[q].w + qym.w), lo_clamp);
                if (act[q]) dst[32 * q] = o;
            }
        }
    }
}

// The tensor map of a volume of the handle's dims at `base` with a (bx, by, 1) box: from the handle's cache, else encoded
// (about a microsecond of host time, which ten sweeps per outer iteration used to pay twice each) and remembered.
// ok = false: the driver cannot encode (no cuTensorMapEncodeTiled) - the caller falls back to the row kernel.
const CUtensorMap *tv_tensor_map(cbct_geometry *g, const float *base, unsigned bx, unsigned by, bool *ok)
{
    static_assert(sizeof(CUtensorMap) <= sizeof(cbct_geometry::TmapSlot::map), "TmapSlot::map holds a CUtensorMap");
    *ok = true;
    for (auto &s : g->tv_tmaps)
        if (s.ptr == base && s.bx == bx && s.by == by) return reinterpret_cast<const CUtensorMap *>(s.map);
    auto &s = g->tv_tmaps[g->tv_tmap_next];
    g->tv_tmap_next = (g->tv_tmap_next + 1) % (int)(sizeof(g->tv_tmaps) / sizeof(g->tv_tmaps[0]));
    const unsigned long long p1 = (unsigned long long)g->nx * sizeof(float), p2 = p1 * g->ny;
    s.ptr = nullptr;
    if (cbct_tensor_map_3d(reinterpret_cast<CUtensorMap *>(s.map), base, g->nx, g->ny, g->nz, p1, p2, bx, by, 1) != CBCT_OK) {
        *ok = false;
        return nullptr;
    }
    s.ptr = base; s.bx = bx; s.by = by;
    return reinterpret_cast<const CUtensorMap *>(s.map);
}

// *launched = false (and CBCT_OK) if the tensor maps cannot be encoded: nothing has been launched, the caller uses tv_rows.cu.
template <int CH, int W>
cbct_status launch_tma(cbct_geometry *g, const float *u_in, const float *gv, float *u_out, float beta, float eps, float dt,
                       int clamp, cudaStream_t st, bool *launched)
{
    using L = TvTmaLayout<CH, W>;
    auto kern = tv_tma_kernel<CH, W>;
    const size_t smem = L::total(g->nx);
    *launched = false;
    const unsigned bx = (unsigned)L::bx(g->nx);
    bool ok = true;
    const CUtensorMap *pu = tv_tensor_map(g, u_in, bx, W + 1, &ok);
    // with g fetched by plain 16-byte loads (kGLdg) the kernel never touches its second map: the first one fills the slot
    const CUtensorMap *pg = (ok && !kGLdg) ? tv_tensor_map(g, gv, bx, W - 1, &ok) : pu;
    if (!ok) return CBCT_OK;
    const CUtensorMap tu = *pu, tg = *pg;
    // kernel attribute and occupancy, cached per instantiation for the whole process; handles may live on different host
    // threads (cbct.h: one handle per thread), so the cache is read and written under a lock
    static std::mutex mtx;
    static int slots_cached = 0;
    static size_t smem_set = 0;
    int slots;
    {
        std::lock_guard<std::mutex> lock(mtx);
        if (!slots_cached || smem > smem_set) {
            CBCT_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            int dev = 0, sms = 0, per_sm = 0;
            CBCT_CUDA(cudaGetDevice(&dev));
            CBCT_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
            CBCT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, 32 * W, smem));
            slots_cached = sms * (per_sm > 0 ? per_sm : 1);
            smem_set = smem;
        }
        slots = slots_cached;
    }
    const int ytiles = (g->ny + W - 2) / (W - 1);
    int zchunk = 8;
    long best = -1;
    for (int zc = 4; zc <= 64; ++zc) {                                          // waves x (planes per chunk + the recomputed one)
        const long ctas = (long)ytiles * ((g->nz + zc - 1) / zc);
        const long cost = ((ctas + slots - 1) / slots) * (zc + 1);
        if (best < 0 || cost < best) { best = cost; zchunk = zc; }
    }
    const double hx = g->hx, hy = g->hy, hz = g->hz;
    dim3 grid(ytiles, (g->nz + zchunk - 1) / zchunk);
    kern<<<grid, 32 * W, smem, st>>>(tu, tg, gv, u_out, g->nx, g->ny, g->nz, (float)(1.0 / (hx * hx)), (float)(1.0 / (hy * hy)),
                                     (float)(1.0 / (hz * hz)), beta, eps * eps, dt, clamp ? 0.f : -INFINITY, zchunk);
    CBCT_LAUNCH_CHECK();
    *launched = true;
    return CBCT_OK;
}
}  // namespace

#ifndef CBCT_TV_TMA_W
#define CBCT_TV_TMA_W 8
#endif

// *done = 1 if this path took the step (nx <= 512, nx % 4 == 0, 16-byte aligned volumes, at least 32 voxels per row, and a
// driver that encodes tensor maps); *done = 0 with CBCT_OK means nothing was launched and the caller takes the row kernel.
cbct_status op_tv_sweep_tma(cbct_geometry *g, const float *u_in, const float *gv, float *u_out, float beta, float eps, float dt,
                            int clamp, cudaStream_t st, int *done)
{
    *done = 0;
    const int nx = g->nx;
    if (nx > 512 || nx < 32 || nx % 4 != 0 || (((uintptr_t)u_in | (uintptr_t)gv | (uintptr_t)u_out) & 15) != 0) return CBCT_OK;
    constexpr int W = CBCT_TV_TMA_W;
    bool launched = false;
    cbct_status rc;
    if (nx <= 128) rc = launch_tma<1, W>(g, u_in, gv, u_out, beta, eps, dt, clamp, st, &launched);
    else if (nx <= 256) rc = launch_tma<2, W>(g, u_in, gv, u_out, beta, eps, dt, clamp, st, &launched);
    else if (nx <= 384) rc = launch_tma<3, W>(g, u_in, gv, u_out, beta, eps, dt, clamp, st, &launched);
    else rc = launch_tma<4, W>(g, u_in, gv, u_out, beta, eps, dt, clamp, st, &launched);
    *done = launched ? 1 : 0;
    return rc;
}
