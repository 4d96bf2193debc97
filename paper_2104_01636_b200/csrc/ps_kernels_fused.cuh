// ps_kernels_fused.cuh -- fused red+black z-marching SOR sweep for sm_100a (TMA + mbarrier).
//
// One launch = one full sweep (red half-sweep, then black half-sweep) in ONE pass over
// memory: p_src, rhs, ax, ay, az are read once and p_dst written once = 48 B per cell-update instead
// of the 96 B the two-pass kernel moves (scheme M2).
//
// Schedule (legal reordering; every value is computed by the same expression from the same
// inputs, so p is bitwise identical to the two-pass kernel and to the oracle):
//   * p ping-pongs: p_src is read-only during the launch, p_dst write-only.
//   * A CTA owns an (x,y) tile and a chunk of z planes and marches in +z.  Step k does
//         red   update of plane k      (needs the OLD black values of planes k-1, k, k+1)
//         black update of plane k-1    (needs the NEW red values of planes k-2, k-1, k)
//     and stores the finished plane k-1 to p_dst.
//   * Black cells on the tile edge need red neighbours owned by other CTAs; instead of an
//     inter-CTA exchange the CTA recomputes red on a one-cell ring around its tile (which needs
//     p_src on a two-cell ring).  The same holds at the two ends of the z chunk.
//
// Data movement: a box of 64 x RB cells (32 column pairs x RB rows; warp = row, lane = pair) of
// each of p, ax, ay, az, rhs per plane is brought into shared memory by the TMA
// (cp.async.bulk.tensor.3d, fp64 tensor maps, mbarrier completion), D planes ahead of use.
// Out-of-bounds box elements are zero-filled by the TMA: exactly the wall convention (a zero
// coefficient on wall faces; a finite neighbour value that meets it).  Periodic z is an explicit
// plane coordinate mod nz.  Each thread reads its pair's coefficients with 128-bit shared loads,
// uses the red cell's half now and carries the black cell's half in registers to the next step;
// p planes stay in shared memory for the x/y neighbour exchange (new red values are written in
// place) -- one __syncthreads per step.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdint>
#include <cstring>

#include "ps_kernels_generic.cuh"

namespace ps {

constexpr int FUSED_RB = 16;       // rows per box = warps per CTA
constexpr int FUSED_D = 3;         // planes in flight ahead of the one being computed
constexpr int FUSED_BOXW = 64;     // cells per box row (32 lanes x 2)
constexpr int FUSED_MAX_TILES = 512;

template <int RB, int D>
struct FusedLayout {
    static constexpr int NC = D + 1;                    // coefficient stages
    static constexpr int NP = D + 4;                    // p planes
    static constexpr int AXW = FUSED_BOXW + 2;          // ax box starts one pair to the left
    static constexpr int P_ELEMS = RB * FUSED_BOXW;
    static constexpr int AX_ELEMS = RB * AXW;
    static constexpr int AY_ELEMS = (RB + 1) * FUSED_BOXW;   // ay box starts one row above
    static constexpr int AZ_ELEMS = RB * FUSED_BOXW;
    static constexpr int RH_ELEMS = RB * FUSED_BOXW;
    static constexpr int C_ELEMS = AX_ELEMS + AY_ELEMS + AZ_ELEMS + RH_ELEMS;
    static constexpr uint32_t P_BYTES = P_ELEMS * 8;
    static constexpr uint32_t C_BYTES = C_ELEMS * 8;
    static constexpr uint32_t AZ_BYTES = AZ_ELEMS * 8;
    static constexpr size_t SMEM_BYTES = (size_t)NP * P_BYTES + (size_t)NC * C_BYTES +
                                         (NP + NC) * 8 + 128 /* alignment slack */;
    static_assert(P_BYTES % 128 == 0 && (AX_ELEMS * 8) % 128 == 0 && (AY_ELEMS * 8) % 128 == 0,
                  "TMA destinations must stay 128-byte aligned");
};

struct FusedParams {
    Grid g;
    int tiles_x, tiles_y, kz;      // kz: planes per z chunk
    const int *xs;                 // tiles_x + 1 interior boundaries (even)
    const int *ys;                 // tiles_y + 1 interior boundaries
    double *p_dst;
    double omega;
};

// ---------------------------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_addr(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    const uint32_t a = smem_addr(bar);
    uint32_t ok = 0;
    do {
        asm volatile(
            "{\n\t.reg .pred q;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 q, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, q;\n\t}"
            : "=r"(ok)
            : "r"(a), "r"(parity)
            : "memory");
    } while (!ok);
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, int x, int y, int z,
                                            uint64_t *bar)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes "
        "[%0], [%1, {%2, %3, %4}], [%5];" ::"r"(smem_addr(dst)),
        "l"((uint64_t)map), "r"(x), "r"(y), "r"(z), "r"(smem_addr(bar))
        : "memory");
}
__device__ __forceinline__ void fence_proxy_async()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ int wrap(int k, int nz)
{
    k %= nz;
    return k < 0 ? k + nz : k;
}

// ---------------------------------------------------------------------------------- the kernel
template <int RB, int D>
__global__ void __launch_bounds__(32 * RB, 1)
ps_fused_sweep_kernel(const __grid_constant__ CUtensorMap mapP, const __grid_constant__ CUtensorMap mapAX,
                      const __grid_constant__ CUtensorMap mapAY, const __grid_constant__ CUtensorMap mapAZ,
                      const __grid_constant__ CUtensorMap mapRH, const FusedParams prm)
{
    using L = FusedLayout<RB, D>;
    extern __shared__ unsigned char smem_raw[];
    unsigned char *base = (unsigned char *)(((uintptr_t)smem_raw + 127) & ~(uintptr_t)127);
    double *sP = (double *)base;                                  // NP planes
    double *sC = sP + (size_t)L::NP * L::P_ELEMS;                 // NC stages: AX | AY | AZ | RH
    uint64_t *barP = (uint64_t *)(sC + (size_t)L::NC * L::C_ELEMS);
    uint64_t *barC = barP + L::NP;

    const int lane = threadIdx.x & 31, r = threadIdx.x >> 5;
    const Grid g = prm.g;

    // ---- tile geometry
    const int xs = prm.xs[blockIdx.x], xe = prm.xs[blockIdx.x + 1];
    const int ys = prm.ys[blockIdx.y], ye = prm.ys[blockIdx.y + 1];
    const int bx = (prm.tiles_x == 1) ? 0 : xs - 2;               // box origin (may be negative)
    const int by = (prm.tiles_y == 1) ? 0 : ys - 2;
    const int ks = blockIdx.z * prm.kz;
    const int ke = min(g.nz, ks + prm.kz);
    const int i0 = bx + 2 * lane, j = by + r;
    const bool in_dom = (i0 >= 0) && (i0 < g.nx) && (j >= 0) && (j < g.ny);
    const bool row_red = in_dom && (j >= ys - 1) && (j < ye + 1);
    const bool red_l = row_red && (i0 >= xs - 1) && (i0 < xe + 1);
    const bool red_r = row_red && (i0 + 1 >= xs - 1) && (i0 + 1 < xe + 1);
    const bool interior = in_dom && (j >= ys) && (j < ye) && (i0 >= xs) && (i0 < xe);

    // shared-memory element offsets inside a p plane
    const int own = r * FUSED_BOXW + 2 * lane;                    // left cell of the pair
    const int outer_l = lane > 0 ? own - 1 : own;                 // x- neighbour of the left cell
    const int outer_r = lane < 31 ? own + 2 : own + 1;            // x+ neighbour of the right cell
    const int dym = (r > 0) ? -FUSED_BOXW : 0, dyp = (r < RB - 1) ? FUSED_BOXW : 0;
    const size_t plane = (size_t)g.nx * g.ny;
    const size_t gofs = (size_t)i0 + (size_t)g.nx * (size_t)(in_dom ? j : 0);

    // ---- barriers
    if (threadIdx.x == 0) {
        for (int q = 0; q < L::NP + L::NC; ++q) mbar_init(barP + q, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // step t = 0 .. T-1 works on plane k = ks - 2 + t; p plane u = 0 .. T is plane ks - 2 + u
    const int T = (ke - ks) + 3;
    auto issue_coef = [&](int t) {        // thread 0 only
        const int slot = t % L::NC, z = wrap(ks - 2 + t, g.nz);
        double *c = sC + (size_t)slot * L::C_ELEMS;
        if (t == 0) {                     // only az of plane ks-2 is needed (azm of the first red)
            mbar_expect_tx(barC + slot, L::AZ_BYTES);
            tma_load_3d(c + L::AX_ELEMS + L::AY_ELEMS, &mapAZ, bx, by, z, barC + slot);
        } else {
            mbar_expect_tx(barC + slot, L::C_BYTES);
            tma_load_3d(c, &mapAX, bx - 2, by, z, barC + slot);
            tma_load_3d(c + L::AX_ELEMS, &mapAY, bx, by - 1, z, barC + slot);
            tma_load_3d(c + L::AX_ELEMS + L::AY_ELEMS, &mapAZ, bx, by, z, barC + slot);
            tma_load_3d(c + L::AX_ELEMS + L::AY_ELEMS + L::AZ_ELEMS, &mapRH, bx, by, z,
                        barC + slot);
        }
    };
    auto issue_p = [&](int u) {           // thread 0 only
        const int slot = u % L::NP;
        mbar_expect_tx(barP + slot, L::P_BYTES);
        tma_load_3d(sP + (size_t)slot * L::P_ELEMS, &mapP, bx, by, wrap(ks - 2 + u, g.nz),
                    barP + slot);
    };
    if (threadIdx.x == 0) {
        for (int t = 0; t < D && t < T; ++t) issue_coef(t);
        for (int u = 0; u <= D && u <= T; ++u) issue_p(u);
    }

    // carried coefficient state (see header): the black cell's half of plane k-1 and az history
    double b_axm = 0.0, b_axp = 0.0, b_aym = 0.0, b_ayp = 0.0, b_rhs = 0.0, az2 = 0.0;
    double2 azprev = make_double2(0.0, 0.0);
    const double omega = prm.omega;

    int C = (j + ks) & 1;                 // column of the pair that is red on plane k (k = ks-2+t)
    for (int t = 0; t < T; ++t, C ^= 1) {
        const int k = ks - 2 + t;
        // everyone is done with step t-1: its coefficient stage and p plane u = t-3 are free
        __syncthreads();
        if (threadIdx.x == 0) {
            if (t + D < T) issue_coef(t + D);
            if (t + D + 1 <= T) issue_p(t + D + 1);
        }
        mbar_wait(barC + t % L::NC, (t / L::NC) & 1);
        if (t == 0) {
            mbar_wait(barP + 0, 0);
            if (T >= 1) mbar_wait(barP + 1 % L::NP, 0);
        } else if (t + 1 <= T) {
            mbar_wait(barP + (t + 1) % L::NP, ((t + 1) / L::NP) & 1);
        }

        const double *c = sC + (size_t)(t % L::NC) * L::C_ELEMS;
        const double2 AZ = *(const double2 *)(c + L::AX_ELEMS + L::AY_ELEMS + own);
        if (t == 0) {                     // prologue: only the az history
            azprev = AZ;
            continue;
        }
        const double2 AX = *(const double2 *)(c + r * L::AXW + 2 * lane + 2);
        const double AXL = c[r * L::AXW + 2 * lane + 1];
        const double2 AYM = *(const double2 *)(c + L::AX_ELEMS + own);
        const double2 AY = *(const double2 *)(c + L::AX_ELEMS + FUSED_BOXW + own);
        const double2 RH = *(const double2 *)(c + L::AX_ELEMS + L::AY_ELEMS + L::AZ_ELEMS + own);

        double *S0 = sP + (size_t)((t) % L::NP) * L::P_ELEMS;            // plane k
        const double *Sp1 = sP + (size_t)((t + 1) % L::NP) * L::P_ELEMS;  // plane k+1
        const double *Sm1 = sP + (size_t)((t + L::NP - 1) % L::NP) * L::P_ELEMS;  // plane k-1
        const double *Sm2 = sP + (size_t)((t + L::NP - 2) % L::NP) * L::P_ELEMS;  // plane k-2

        const int oc = own + C;           // this step's column in the pair
        const double axm = C ? AX.x : AXL, axp = C ? AX.y : AX.x;
        const double aym = C ? AYM.y : AYM.x, ayp = C ? AY.y : AY.x;
        const double azp = C ? AZ.y : AZ.x, azm = C ? azprev.y : azprev.x;
        const double rh = C ? RH.y : RH.x;
        const double pm1c = Sm1[oc];      // old black of plane k-1 (z- neighbour of the red cell)

        // ---- red update of plane k
        double rnew = 0.0;
        if (C ? red_r : red_l) {
            const double pxm = C ? S0[own] : S0[outer_l];
            const double pxp = C ? S0[outer_r] : S0[own + 1];
            rnew = sor_update(axm, axp, aym, ayp, azm, azp, pxm, pxp, S0[oc + dym], S0[oc + dyp],
                              pm1c, Sp1[oc], S0[oc], rh, omega);
            S0[oc] = rnew;                // visible to the neighbours after the next barrier
        }
        // ---- black update of plane k-1 (same column), then store the finished pair
        if (interior && t >= 3) {
            const double pxm = C ? Sm1[own] : Sm1[outer_l];
            const double pxp = C ? Sm1[outer_r] : Sm1[own + 1];
            const double bnew = sor_update(b_axm, b_axp, b_aym, b_ayp, az2, azm, pxm, pxp,
                                           Sm1[oc + dym], Sm1[oc + dyp], Sm2[oc], rnew, pm1c, b_rhs,
                                           omega);
            const double other = Sm1[own + (C ^ 1)];       // red value of plane k-1 (this thread's)
            const double2 outv = C ? make_double2(other, bnew) : make_double2(bnew, other);
            *(double2 *)(prm.p_dst + gofs + plane * (size_t)wrap(k - 1, g.nz)) = outv;
        }
        // ---- carry the other column's half of plane k to the next step
        b_axm = C ? AXL : AX.x;
        b_axp = C ? AX.x : AX.y;
        b_aym = C ? AYM.x : AYM.y;
        b_ayp = C ? AY.x : AY.y;
        b_rhs = C ? RH.x : RH.y;
        az2 = C ? azprev.x : azprev.y;
        azprev = AZ;
        fence_proxy_async();              // generic writes to S0 before the TMA reuses the slot
    }
}

// ---------------------------------------------------------------------------------- host side
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *,
                                  const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                                  const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct FusedPlan {
    int sm_count;
    bool ok;
    int tiles_x, tiles_y, kz, tiles_z;
    int *d_xs, *d_ys;               // device copies of the tile boundaries
    EncodeTiledFn encode;
    // tensor-map cache: index 0..4 = p, ax, ay, az, rhs
    const void *cached_ptr[5];
    CUtensorMap maps[5];
};

inline bool fused_shape_ok(const Grid &g)
{
    return (g.nx % 2 == 0) && g.nx >= 4 && g.ny >= 1 && g.nz >= 2 && (g.nz % 2 == 0) &&
           ((size_t)g.nx * 8 % 16 == 0);
}

// Split [0,n) into tiles whose interior fits the box: a box of `box` cells needs a halo of 2 on
// every side that is not a wall.  Boundaries are multiples of `align`.
inline int make_tiles(int n, int box, int align, int *out /* FUSED_MAX_TILES + 1 */)
{
    if (n <= box) { out[0] = 0; out[1] = n; return 1; }
    for (int t = 2; t <= FUSED_MAX_TILES; ++t) {
        const int cap_end = box - 2, cap_mid = box - 4;
        if ((long long)cap_mid * (t - 2) + 2LL * cap_end < n) continue;
        // even split, remainder handed out from the two ends inwards
        int w[FUSED_MAX_TILES];
        const int basew = (n / t) / align * align;
        int rem = n - basew * t;
        for (int q = 0; q < t; ++q) w[q] = basew;
        for (int q = 0; rem > 0; ++q) {
            const int idx = (q & 1) ? t - 1 - (q >> 1) % t : (q >> 1) % t;
            w[idx] += align;
            rem -= align;
        }
        bool good = true;
        for (int q = 0; q < t; ++q) {
            const int cap = (q == 0 || q == t - 1) ? cap_end : cap_mid;
            if (w[q] > cap || w[q] <= 0) good = false;
        }
        if (!good) continue;
        out[0] = 0;
        for (int q = 0; q < t; ++q) out[q + 1] = out[q] + w[q];
        return t;
    }
    return -1;
}

inline cudaError_t fused_plan_init(FusedPlan *pl, const Grid &g, int sm_count)
{
    memset(pl, 0, sizeof *pl);
    pl->sm_count = sm_count;
    if (!fused_shape_ok(g)) return cudaSuccess;
    int hx[FUSED_MAX_TILES + 1], hy[FUSED_MAX_TILES + 1];
    pl->tiles_x = make_tiles(g.nx, FUSED_BOXW, 2, hx);
    pl->tiles_y = make_tiles(g.ny, FUSED_RB, 1, hy);
    if (pl->tiles_x < 0 || pl->tiles_y < 0) return cudaSuccess;      // too wide: not available
    // z chunks: enough CTAs for ~4 waves of the device, chunks of at least 16 planes
    const long long per_plane = (long long)pl->tiles_x * pl->tiles_y;
    int tz = (int)((4LL * sm_count + per_plane - 1) / per_plane);
    if (tz < 1) tz = 1;
    int kz = (g.nz + tz - 1) / tz;
    if (kz < 16) kz = 16;
    if (kz > g.nz) kz = g.nz;
    kz = (kz + 1) & ~1;                                               // even: parity bookkeeping
    pl->kz = kz;
    pl->tiles_z = (g.nz + kz - 1) / kz;
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess) return e;
    if (qres != cudaDriverEntryPointSuccess || !fn) return cudaErrorNotSupported;
    pl->encode = (EncodeTiledFn)fn;
    e = cudaMalloc((void **)&pl->d_xs, (pl->tiles_x + 1 + pl->tiles_y + 1) * sizeof(int));
    if (e != cudaSuccess) return e;
    pl->d_ys = pl->d_xs + pl->tiles_x + 1;
    e = cudaMemcpy(pl->d_xs, hx, (pl->tiles_x + 1) * sizeof(int), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return e;
    e = cudaMemcpy(pl->d_ys, hy, (pl->tiles_y + 1) * sizeof(int), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(ps_fused_sweep_kernel<FUSED_RB, FUSED_D>,
                             cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)FusedLayout<FUSED_RB, FUSED_D>::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    pl->ok = true;
    return cudaSuccess;
}

inline void fused_plan_destroy(FusedPlan *pl)
{
    if (pl->d_xs) cudaFree(pl->d_xs);
    pl->d_xs = pl->d_ys = nullptr;
    pl->ok = false;
}

inline cudaError_t fused_map(FusedPlan &pl, int which, const Grid &g, const void *ptr, int boxw,
                             int boxh)
{
    if (pl.cached_ptr[which] == ptr) return cudaSuccess;
    const cuuint64_t dims[3] = {(cuuint64_t)g.nx, (cuuint64_t)g.ny, (cuuint64_t)g.nz};
    const cuuint64_t strides[2] = {(cuuint64_t)g.nx * 8, (cuuint64_t)g.nx * g.ny * 8};
    const cuuint32_t box[3] = {(cuuint32_t)boxw, (cuuint32_t)boxh, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = pl.encode(&pl.maps[which], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3,
                                 const_cast<void *>(ptr), dims, strides, box, estr,
                                 CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                 CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                                 CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
    pl.cached_ptr[which] = ptr;
    return cudaSuccess;
}

// One fused sweep p_src -> p_dst.  `want` sweeps requested; *did = sweeps this launch performs.
inline cudaError_t launch_fused(FusedPlan &pl, const Grid &g, const double *ax, const double *ay,
                                const double *az, const double *rhs, const double *p_src,
                                double *p_dst, double omega, int want, cudaStream_t stream, int *did)
{
    (void)want;
    *did = 0;
    if (!pl.ok) return cudaErrorNotSupported;
    using L = FusedLayout<FUSED_RB, FUSED_D>;
    cudaError_t e;
    if ((e = fused_map(pl, 0, g, p_src, FUSED_BOXW, FUSED_RB)) != cudaSuccess) return e;
    if ((e = fused_map(pl, 1, g, ax, L::AXW, FUSED_RB)) != cudaSuccess) return e;
    if ((e = fused_map(pl, 2, g, ay, FUSED_BOXW, FUSED_RB + 1)) != cudaSuccess) return e;
    if ((e = fused_map(pl, 3, g, az, FUSED_BOXW, FUSED_RB)) != cudaSuccess) return e;
    if ((e = fused_map(pl, 4, g, rhs, FUSED_BOXW, FUSED_RB)) != cudaSuccess) return e;
    FusedParams prm;
    prm.g = g;
    prm.tiles_x = pl.tiles_x;
    prm.tiles_y = pl.tiles_y;
    prm.kz = pl.kz;
    prm.xs = pl.d_xs;
    prm.ys = pl.d_ys;
    prm.p_dst = p_dst;
    prm.omega = omega;
    const dim3 grid(pl.tiles_x, pl.tiles_y, pl.tiles_z);
    ps_fused_sweep_kernel<FUSED_RB, FUSED_D><<<grid, 32 * FUSED_RB, L::SMEM_BYTES, stream>>>(
        pl.maps[0], pl.maps[1], pl.maps[2], pl.maps[3], pl.maps[4], prm);
    *did = 1;
    return cudaGetLastError();
}

}  // namespace ps
