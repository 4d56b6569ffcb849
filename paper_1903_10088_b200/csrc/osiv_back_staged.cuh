// osiv_back_staged.cuh -- K2 of the quarter-turn path with its per-block inputs staged in shared memory
// (include/osiv.h).  Same arithmetic as k_back<MODE, 4, 1, 0> (osiv_kernels.cuh): matched gather
// backprojection g = A_S^T r ("estimation"), step rule Eq. 4-5, TV gradient (C8),
// Eq. 3 update with mu >= 0, best-image copy.
//
// Why a second K2.  ncu on k_back at config 3 (profiles/r2a): 63 % of its executed instructions are start-up, interval
// fetch/decode and epilogue, its candidate loop runs at the L1 data-pipe wavefront limit (two 16-byte gathers per
// candidate and thread) and every trip waits for an L2 round trip.  Here
//   * a block owns a compact rectangle of the base quadrant (about 20 x 22 pixels; table `BackSArgs::regions`, which
//     travels in the kernel parameters: a block reads its entry from the constant bank, not behind an L2 round trip),
//     so the channels its tiles can see in one view form ONE short window of W channels;
//   * everything constant a block needs for one subset -- per view the window of the ray table, compressed to 8 bytes
//     per ray {k, g0} (one of alpha, beta is exactly 1 after a sign flip, which of them is a per-window flag; the
//     half-width follows from k), and the block's row of candidate intervals -- lies CONTIGUOUSLY in a per-subset
//     "blob" (k_build_blob, once per handle and subset count) and reaches shared memory with ONE bulk copy
//     (cp.async.bulk + mbarrier: no registers, no waiting threads), issued before the dependent-launch wait; the
//     residual windows (K1's output) follow with one bulk copy per view right after the wait, spread over the warps
//     (a single warp issuing 120 small copies took 5 us; the copy engine serves a request in about 25 cycles), one
//     mbarrier per base view, so the walk starts as soon as the first view has landed; the next subset's blob is
//     prefetched into L2 by the same launch;
//   * a thread's tile is 4 x 2 pixels (x 4 rotations = 32 accumulators as 16 FFMA2 pairs): 35 % fewer candidate loads
//     per pixel than 2 x 2 tiles; a candidate costs one 8-byte and one 16-byte shared-memory load (the walk is bound
//     by shared-memory wavefronts), a trip one 16-bit load and a handful of integer instructions;
//   * everything of the epilogue that does not need the sums (the 3 x 3 neighbourhood of orbit float4s, the TV gradient
//     of all four rotated pixels) is done before the walk, while the copies are in flight; the first warp out of the
//     walk evaluates the step rule from inputs that went to shared memory by cp.async during the walk; after the block
//     barrier a thread only sums the eight view shares of one base pixel, updates its four rotations and stores.
// The general kernel k_back stays the path for everything this one does not take (NS = 1, pairs of slices, stacks,
// grids whose side is not a multiple of 8, fans of 90 degrees or more, windows that do not fit).
#pragma once
#include "osiv_kernels.cuh"

namespace osiv {

constexpr int BS_TX = 4, BS_TY = 2, BS_PX = 8;       // pixels per thread tile
constexpr int BS_SHARES = 8;                         // view shares per tile: quarter turn (4) x 2 sub-shares
constexpr int BS_MAX_REGIONS = 1024;                 // blocks per slice (regions of the base quadrant)
constexpr int BS_MAX_TPB = 64;                       // tile slots per block (threads = 8 x slots = 512: 16 warps, four per scheduler with 128
                                                     // registers each; a 17th warp would put five on one scheduler's 16K registers: 96)
constexpr int BS_MAX_JR = 16;                        // base views staged per round = mbarriers
constexpr int BS_RED_PITCH = BS_PX + 1;              // float4 per (share, tile) row of the reduction buffer: odd, conflict-free
constexpr int BS_RCH = 8;                            // residual chunks (16 bytes) a thread fetches per round: 4 * JR * W <= 8 * threads
constexpr int BS_DPK = 8;                            // monitor partials per lane of the step-rule warp: K1 blocks per slice <= 256
constexpr int BS_HDR_BYTES = 2560;                   // mbarrier, step/improved words, ticket (first 256 bytes), then the slice's monitor
                                                     // partials [32 * BS_DPK] doubles and its SliceState, in front of the staging area
constexpr int BS_PARAM_REGIONS = 160;                // regions that travel in the kernel parameters (constant bank) instead of a table

struct BackSArgs {
    BackArgs b;                            // geometry, residuals, images, state, step-rule parameters (as for k_back)
    const int4* regions;                   // [nblk] {tx0 | ty0 << 16, w | h << 16, ceil(2^32 / w), 0} in tiles of 4 x 2 pixels
    const unsigned char* blob;             // [M][nblk][V_S] slots of slot_c bytes: {c0, orientation, 0, 0} (16 bytes),
                                           // ray window [W] {k, g0}, interval row [tpbp] u16 (first candidate | count << 8)
    int nblk, tpbp;                        // blocks per slice, tile slots per block (multiple of 32)
    unsigned tpbp_magic;
    int W;                                 // window length in channels (all blocks, all views; even)
    int JR, nrounds;                       // base views staged per round, rounds
    unsigned W_magic;
    int SP;                                // residual slots fetched per pass = threads / W
    int slot_c;                            // 16 + W * 8 + tpbp * 2
    float hka, hkb;                        // half-width of a ray's trapezoid = |k| * hka + hkb (exact chord: 1/2, 1/2; Joseph: 0, 1)
    // the same table in the kernel parameters when nblk <= BS_PARAM_REGIONS: a block learns its region from the constant
    // bank instead of with an L2 round trip at the head of its start-up path (its neighbourhood loads depend on it)
    int4 regions_c[BS_PARAM_REGIONS];
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, int bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, int parity) {
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
// global -> shared bulk copy (16-byte aligned, size a multiple of 16), completion counted in bytes on `bar`
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, int bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// 8-byte asynchronous copy global -> shared (the monitor partials travel during the walk, no registers held)
__device__ __forceinline__ void cp_async8(uint32_t dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

__device__ __forceinline__ void bulk_prefetch_l2(const void* src, int bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}

// Ray-table entry {alpha, beta, g0, hk} -> {k, g0} with the unit coefficient made +1 by a sign flip (|q| does not see
// it): x-unit (returns true): alpha = 1, beta = k; y-unit: alpha = k, beta = 1.  The all-zero slack entries behind the
// table become a ray that misses everything.
__device__ __forceinline__ bool ray_to8(const float4 r, float2& e) {
    if (fabsf(r.y) == 1.f) { e = make_float2(r.x * r.y, r.z * r.y); return false; }
    if (fabsf(r.x) == 1.f) { e = make_float2(r.y * r.x, r.z * r.x); return true; }
    e = make_float2(0.f, 1e30f);
    return true;
}

// The eight chord weights (over h) of candidate ray {k, g0} for the 4 x 2 tile whose first pixel has centred indices
// (xc0, yc0); pixel p = ty * 4 + tx; ORI 0: x-unit, 1: y-unit, 2: decided by xu.  All three evaluate
// q = alpha*xc + beta*yc + g0 with the same float operations as fmaf(alpha, xc0, fmaf(beta, yc0, g0)) and the chain
// q(tx+1) = q(tx) + alpha, q(ty+1) = q(ty) + beta, so they agree bit for bit, and the set-up kernel and the walk both
// call this: a candidate outside the tabulated support contributes exactly 0.
template <int ORI>
__device__ __forceinline__ void bs_weights(const float2 e, bool xu, float xc0, float yc0, float hka, float hkb, float (&w)[BS_PX]) {
    const float k = e.x;
    const float hk = fmaf(fabsf(k), hka, hkb);
    float q[BS_PX];
    if (ORI == 0 || (ORI == 2 && xu)) {
        q[0] = xc0 + fmaf(k, yc0, e.y);
        q[1] = q[0] + 1.f; q[2] = q[1] + 1.f; q[3] = q[2] + 1.f;
#pragma unroll
        for (int p = 0; p < 4; ++p) q[4 + p] = q[p] + k;
    } else {
        q[0] = fmaf(k, xc0, yc0 + e.y);
        q[1] = q[0] + k; q[2] = q[1] + k; q[3] = q[2] + k;
#pragma unroll
        for (int p = 0; p < 4; ++p) q[4 + p] = q[p] + 1.f;
    }
#pragma unroll
    for (int p = 0; p < BS_PX; ++p) w[p] = __saturatef(hk - fabsf(q[p]));
}

// region of block b and the tile of slot i in it: origin (x0, y0) of the 4 x 2 tile in the base quadrant
__device__ __forceinline__ bool bs_tile(const int4 reg, int i, int& x0, int& y0) {
    const int tx0 = reg.x & 0xffff, ty0 = reg.x >> 16, w = reg.y & 0xffff, h = reg.y >> 16;
    const int iy = fastdiv(i, (unsigned)reg.z), ix = i - iy * w;
    x0 = (tx0 + ix) * BS_TX;
    y0 = (ty0 + iy) * BS_TY;
    return i < w * h;
}

// A0 for the staged K2, once per handle: for every (table view v, block b) the exact support [first, first + count) of
// every tile of the block (first and last channel for which bs_weights gives a non-zero weight to one of its pixels),
// the block's window start = the smallest `first`, and the largest window length and count over everything
// (maxima[0], maxima[1]; the host sizes W from them).  grid (nblk, V), tpbp threads.
__global__ void __launch_bounds__(BS_MAX_TPB) k_build_staged(DevGeom g, float tile_hw, float hka, float hkb, const int4* __restrict__ regions, int nblk, int tpbp,
                                                             unsigned short* __restrict__ itab, int* __restrict__ bwin, int* __restrict__ maxima) {
    const int b = blockIdx.x, v = blockIdx.y, i = threadIdx.x;
    __shared__ int s_lo, s_hi, s_cnt;
    if (i == 0) { s_lo = 1 << 30; s_hi = 0; s_cnt = 0; }
    __syncthreads();
    int x0, y0;
    const bool active = bs_tile(__ldg(&regions[b]), i, x0, y0);
    int first = -1, last = -1, c_lo = 0;
    if (active) {
        // loose interval: every ray with a non-zero weight passes within the tile's radius of its centre
        const float X = ((float)x0 - g.cx + 0.5f * (BS_TX - 1)) * g.pixel, Y = ((float)y0 - g.cy + 0.5f * (BS_TY - 1)) * g.pixel;
        const float2 cs = __ldg(&g.views[v]);
        const float along = g.sad - fmaf(X, cs.x, Y * cs.y);
        const float perp = fmaf(X, cs.y, -Y * cs.x);
        const float rinv = __fdividef(1.f, along);
        const float gam = atanf(perp * rinv);
        const float cstar = fmaf(gam, g.inv_dgamma, g.c_center);
        const float hw = fmaf(tile_hw, rinv, 0.05f);
        c_lo = min(max(0, (int)ceilf(cstar - hw)), g.C);
        const int c_hi = min(g.C - 1, (int)floorf(cstar + hw));
        const float xc0 = (float)x0 - g.cx, yc0 = (float)y0 - g.cy;
        for (int c = c_lo; c <= c_hi; ++c) {
            float w[BS_PX];
            float2 e;
            const bool xu = ray_to8(__ldg(&g.rays[(size_t)v * g.C + c]), e);
            bs_weights<2>(e, xu, xc0, yc0, hka, hkb, w);
            bool any = false;
#pragma unroll
            for (int p = 0; p < BS_PX; ++p) any = any || w[p] > 0.f;
            if (any) { if (first < 0) first = c; last = c; }
        }
        if (first >= 0) { atomicMin(&s_lo, first); atomicMax(&s_hi, last + 1); atomicMax(&s_cnt, last - first + 1); }
    }
    __syncthreads();
    const int c0 = s_hi > 0 ? s_lo : 0;
    unsigned short e = 0;
    if (first >= 0) {
        const int rel = first - c0, cnt = last - first + 1;
        e = (rel < 256 && cnt < 256) ? (unsigned short)(rel | (cnt << 8)) : (unsigned short)0xffff;     // 0xffff: does not fit (host checks maxima)
    }
    itab[((size_t)v * nblk + b) * tpbp + i] = e;
    if (i == 0) {
        bwin[(size_t)v * nblk + b] = c0;
        if (s_hi > 0) { atomicMax(&maxima[0], s_hi - s_lo); atomicMax(&maxima[1], s_cnt); }
    }
}

// The blob of M subsets (once per handle and M): slot (m, b, jb * 4 + qt) = table view v = m + (jb + qt * V_S/4) * M
// seen from block b: header {c0, orientation, 0, 0}, the window's rays as {k, g0}, the block's interval row.
// orientation: 0 = every ray of the window is x-unit, 1 = y-unit, 2 + 2 * s + o = the first s rays have orientation o
// (0: x-unit), the rest the other one (a fan below 90 degrees changes orientation at most once per view).
// grid (nblk, V_S, M), 128 threads.
__global__ void __launch_bounds__(128) k_build_blob(DevGeom g, int M, int VS, int nblk, int tpbp, int W, int slot_c,
                                                    const unsigned short* __restrict__ itab, const int* __restrict__ bwin,
                                                    unsigned char* __restrict__ blob) {
    const int b = blockIdx.x, slot = blockIdx.y, m = blockIdx.z, t = threadIdx.x;
    const int VSb = VS >> 2, jb = slot >> 2, qt = slot & 3;
    const int v = m + (jb + qt * VSb) * M;
    const int c0 = __ldg(&bwin[(size_t)v * nblk + b]);
    unsigned char* dst = blob + (((size_t)m * nblk + b) * VS + slot) * slot_c;
    __shared__ int s_sw;
    float2 e0;
    const bool o0 = ray_to8(__ldg(&g.rays[(size_t)v * g.C + c0]), e0);
    if (t == 0) s_sw = 1 << 30;
    __syncthreads();
    for (int r = t; r < W; r += 128) {
        float2 e = make_float2(0.f, 1e30f);                 // past the view's last channel: a ray that misses everything
        if (c0 + r < g.C) {
            const bool xu = ray_to8(__ldg(&g.rays[(size_t)v * g.C + c0 + r]), e);
            if (xu != o0) atomicMin(&s_sw, r);
        }
        reinterpret_cast<float2*>(dst + 16)[r] = e;
    }
    for (int r = t; r < tpbp; r += 128)
        reinterpret_cast<unsigned short*>(dst + 16 + (size_t)W * 8)[r] = __ldg(&itab[((size_t)v * nblk + b) * tpbp + r]);
    __syncthreads();
    if (t == 0) {
        const int sw = s_sw;
        reinterpret_cast<int4*>(dst)[0] = make_int4(c0, sw >= W ? (o0 ? 0 : 1) : 2 + 2 * sw + (o0 ? 0 : 1), 0, 0);
    }
}

// the candidates [rel, rel + n) of one trip against the thread's tile; two per step, then the odd one
template <int ORI>
__device__ __forceinline__ void bs_walk(const float2* __restrict__ rp, const float4* __restrict__ vp, int n, int rel, int sw, bool o_first_x,
                                        float xc0, float yc0, float hka, float hkb, uint64_t (&acc)[2][BS_PX]) {
    int u = 0;
#pragma unroll 1
    for (; u + 1 < n; u += 2) {
        const float2 e0 = rp[u], e1 = rp[u + 1];
        const float4 v0 = vp[u], v1 = vp[u + 1];
        float w0[BS_PX], w1[BS_PX];
        bs_weights<ORI>(e0, (rel + u < sw) == o_first_x, xc0, yc0, hka, hkb, w0);
        bs_weights<ORI>(e1, (rel + u + 1 < sw) == o_first_x, xc0, yc0, hka, hkb, w1);
        const uint64_t a0 = pack2(v0.x, v0.y), b0 = pack2(v0.z, v0.w), a1 = pack2(v1.x, v1.y), b1 = pack2(v1.z, v1.w);
#pragma unroll
        for (int p = 0; p < BS_PX; ++p) {
            ffma2(acc[0][p], a0, w0[p]); ffma2(acc[1][p], b0, w0[p]);
            ffma2(acc[0][p], a1, w1[p]); ffma2(acc[1][p], b1, w1[p]);
        }
    }
    if (u < n) {
        const float2 e0 = rp[u];
        const float4 v0 = vp[u];
        float w0[BS_PX];
        bs_weights<ORI>(e0, (rel + u < sw) == o_first_x, xc0, yc0, hka, hkb, w0);
        const uint64_t a0 = pack2(v0.x, v0.y), b0 = pack2(v0.z, v0.w);
#pragma unroll
        for (int p = 0; p < BS_PX; ++p) { ffma2(acc[0][p], a0, w0[p]); ffma2(acc[1][p], b0, w0[p]); }
    }
}

// ------------------------------------------------------------------------------------------------
// The kernel.  Threads: 8 * tpbp walkers (share q = t / tpbp: quarter turn q & 3, sub-share q >> 2; tile slot
// i = t % tpbp); warp 0 also evaluates the step rule.  Shared memory: header (mbarriers, step), the round's constant slots
// (one bulk copy out of the blob), the round's residual windows [slot][W] float4, the reduction buffer
// [8 shares][tpbp][9] float4.  One mbarrier: the blob part.
// ------------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(BS_SHARES * BS_MAX_TPB, 1) k_back_staged(const BackSArgs sa) {
    const BackArgs& a = sa.b;
    const DevGeom& g = a.g;
    const int t = threadIdx.x, lane = t & 31, s = blockIdx.z, b = blockIdx.x;
    const int tpbp = sa.tpbp;
    const bool first_warp = t < 32; (void)first_warp;     // (timeline build)
    OSIV_TL(a.iter, 1, 0, false);
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t sm0 = smem_u32(smem);
    float* s_step = reinterpret_cast<float*>(smem + 16);
    int* s_ticket = reinterpret_cast<int*>(smem + 32);                          // first warp out of the walk        // [0] step = lambda * tau, [1] improved (as int)
    const int VSb = a.VS >> 2, N = g.nx, JR = sa.JR, W = sa.W;
    unsigned char* cst = smem + BS_HDR_BYTES;                                    // constant slots of the round
    float4* rst = reinterpret_cast<float4*>(cst + (size_t)JR * 4 * sa.slot_c);    // residual windows of the round
    float4* red = rst + (size_t)JR * 4 * W;
    const int msub = a.subset < 0 ? 0 : a.subset;
    const unsigned char* blob = sa.blob + ((size_t)msub * sa.nblk + b) * a.VS * sa.slot_c;   // this block's slots of this subset
    const float* res_s = a.res + (size_t)s * a.VS * a.Cp;

    if (t == 0) {
        mbar_init(sm0, 1);
        mbar_fence_init();
        // round 0's constants: one bulk copy, before anything else
        const int bytes = min(JR, VSb) * 4 * sa.slot_c;
        mbar_expect_tx(sm0, bytes);
        bulk_g2s(sm0 + BS_HDR_BYTES, blob, bytes, sm0);
        *s_ticket = 0;
        // the next subset's constants towards L2 (a cycle through all subsets' blobs does not stay there)
        if (MODE == 1 && a.M > 1 && a.subset >= 0) {
            const int mn = a.subset + 1 == a.M ? 0 : a.subset + 1;
            bulk_prefetch_l2(sa.blob + ((size_t)mn * sa.nblk + b) * a.VS * sa.slot_c, bytes);
        }
    }
    // The residual windows of a round are fetched by all threads with plain 16-byte loads (a bulk copy per window landed
    // a microsecond and more after its issue).  Thread t = s0 * W + r takes channel r of slots s0, s0 + SP, s0 + 2 SP, ...
    // (SP = #threads / W slots per pass); the window starts come out of the blob's slot headers in global memory and the
    // element offsets are worked out before the wait, so that after it a thread only issues its loads.
    const int SP = sa.SP, s0 = fastdiv(t, sa.W_magic), r0 = t - s0 * W;
    int roff[BS_RCH];                                     // float4 index of this thread's chunk in pass n, or -1
    auto load_c0 = [&](int j0, int nj) {
#pragma unroll
        for (int n = 0; n < BS_RCH; ++n) {
            const int slot = n * SP + s0;
            const bool ok = s0 < SP && slot < nj * 4;
            const int c0 = __ldg(reinterpret_cast<const int*>(blob + (size_t)(j0 * 4 + (ok ? slot : 0)) * sa.slot_c));
            roff[n] = ok ? (j0 + (slot >> 2)) * a.Cp + c0 + r0 : -1;
            OSIV_CHECK(!ok || (c0 >= 0 && c0 + W <= a.Cp && (long long)(roff[n] + 1) * 4 <= (long long)a.VS * a.Cp), 6);
        }
    };
    auto load_res = [&](float4 (&rv)[BS_RCH]) {
#pragma unroll
        for (int n = 0; n < BS_RCH; ++n)
            if (roff[n] >= 0) rv[n] = __ldcg(reinterpret_cast<const float4*>(res_s) + roff[n]);
    };
    auto store_res = [&](const float4 (&rv)[BS_RCH]) {
#pragma unroll
        for (int n = 0; n < BS_RCH; ++n)
            if (roff[n] >= 0) rst[(n * SP + s0) * W + r0] = rv[n];
    };
    load_c0(0, min(JR, VSb));
    const int4 reg = sa.nblk <= BS_PARAM_REGIONS ? sa.regions_c[b] : sa.regions[b];
    // walk role: tile slot i, share q
    const int q = fastdiv(t, sa.tpbp_magic), i = t - q * tpbp;
    int x0, y0;
    const bool active = bs_tile(reg, i, x0, y0);
    const float xc0 = (float)x0 - g.cx, yc0 = (float)y0 - g.cy;
    const int quarter = q & 3, ss = q >> 2;
    // finishing role: base pixel pe of tile slot ie, all four rotations
    const int ie = t >> 3, pe = t & 7;
    int ex0, ey0;
    const bool fin = bs_tile(reg, ie, ex0, ey0);
    const int px = ex0 + (pe & 3), py = ey0 + (pe >> 2);
    OSIV_TL(a.iter, 1, 7, false);

    // the 3 x 3 neighbourhood of orbit float4s of mu(n) around P: requested now, used after the copies are on their way
    // (mu(n) is complete: the predecessor K1 released this launch only after its own wait for the K2 that wrote it)
    float4 E[3][3];
    if (MODE == 1 && fin) {
        const float4* Q = reinterpret_cast<const float4*>(a.img) + (size_t)s * g.img_elems;
#pragma unroll
        for (int dy = 0; dy < 3; ++dy)
#pragma unroll
            for (int dx = 0; dx < 3; ++dx) E[dy][dx] = __ldg(Q + (size_t)((py + dy - 1 + PADR) * g.pitch + PAD + px + dx - 1));
    }
    // (no block barrier here: the mbarrier thread 0 has initialised is first touched by the others behind the barrier that
    // follows the residual stores, and a barrier in the start-up path would make every warp wait for thread 0's set-up)
    OSIV_TL(a.iter, 1, 1, false);
    pdl_wait();                                           // the residuals and the monitor partials are the previous launch's output
    pdl_launch_next();
    OSIV_TL(a.iter, 1, 2, false);
    float4 rv[BS_RCH];
    load_res(rv);
    // A3's inputs (K1's monitor partials of this slice, the state after the previous iteration) set out for shared memory
    // now: the warp that evaluates the step rule after its walk then finds them there instead of behind a round trip
    double* dp_s = reinterpret_cast<double*>(smem + 256);
    double* st_s = dp_s + 32 * BS_DPK;
    if (MODE == 1 && first_warp) {
#pragma unroll
        for (int k = 0; k < BS_DPK; ++k)
            if (lane + 32 * k < a.nparts) cp_async8(smem_u32(dp_s + lane + 32 * k), &a.dparts[(size_t)s * a.nparts + lane + 32 * k]);
        if (lane < (int)(sizeof(SliceState) / 8)) cp_async8(smem_u32(st_s + lane), reinterpret_cast<const double*>(&a.state_in[s]) + lane);
        cp_async_commit();
    }
    if (first_warp) OSIV_TL(a.iter, 1, 10, true);

    // ---- while the loads fly: A5 for R^k P, k = 0..3; then the windows go to shared memory; then A3 in warp 0
    float cur[4] = {0.f, 0.f, 0.f, 0.f}, tv[4] = {0.f, 0.f, 0.f, 0.f};
    if (MODE == 1) {
        if (fin) {
            if (px > 0 && py > 0) {                       // P lies in the base quadrant: off the image border
                orbit_tv_inner<0>(E, a.eps2, cur[0], tv[0]);
                orbit_tv_inner<1>(E, a.eps2, cur[1], tv[1]);
                orbit_tv_inner<2>(E, a.eps2, cur[2], tv[2]);
                orbit_tv_inner<3>(E, a.eps2, cur[3], tv[3]);
            } else {
                orbit_tv<0>(E, px, py, N, a.eps2, cur[0], tv[0]);
                orbit_tv<1>(E, px, py, N, a.eps2, cur[1], tv[1]);
                orbit_tv<2>(E, px, py, N, a.eps2, cur[2], tv[2]);
                orbit_tv<3>(E, px, py, N, a.eps2, cur[3], tv[3]);
            }
        }
    }
    OSIV_TL(a.iter, 1, 9, true);
    store_res(rv);
    OSIV_TL(a.iter, 1, 12, true);
    if (MODE == 1 && first_warp) cp_async_wait_all();
    __syncthreads();                                      // residual windows (and the step rule's inputs) in place
    OSIV_TL(a.iter, 1, 11, true);

    uint64_t acc[2][BS_PX];                               // [h][p]: components (2h, 2h+1) of the orbit's residuals for pixel p
#pragma unroll
    for (int h = 0; h < 2; ++h)
#pragma unroll
        for (int p = 0; p < BS_PX; ++p) acc[h][p] = 0ull;

    const int nsub = BS_SHARES >> 2;
#pragma unroll 1
    for (int round = 0; round < sa.nrounds; ++round) {
        const int j0 = round * JR, nj = min(JR, VSb - j0);
        const int parity = round & 1;
        if (round > 0) {
            __syncthreads();                              // everybody has left the previous round's slots
            if (t == 0) {
                fence_proxy_async();
                mbar_expect_tx(sm0, nj * 4 * sa.slot_c);
                bulk_g2s(sm0 + BS_HDR_BYTES, blob + (size_t)j0 * 4 * sa.slot_c, nj * 4 * sa.slot_c, sm0);
            }
            load_c0(j0, nj);
            load_res(rv);
            store_res(rv);
            __syncthreads();
        }
        {
            while (!mbar_try_wait(sm0, parity)) {}
            if (round == 0) OSIV_TL(a.iter, 1, 13, true);
#pragma unroll 1
            for (int jl = ss; jl < nj; jl += nsub) {
                const int slot = jl * 4 + quarter;
                const unsigned char* sp = cst + (size_t)slot * sa.slot_c;
                const int ori = reinterpret_cast<const int*>(sp)[1];
                const unsigned e = reinterpret_cast<const unsigned short*>(sp + 16 + W * 8)[i];
                const int cnt = active ? (int)(e >> 8) : 0, rel = e & 0xff;
                const int n = __reduce_max_sync(0xffffffffu, cnt);
                OSIV_CHECK(e != 0xffffu && rel + n <= W && slot < JR * 4, 7);
                const float2* rp = reinterpret_cast<const float2*>(sp + 16) + rel;
                const float4* vp = rst + (size_t)slot * W + rel;
                // the warp walks max-over-lanes candidates in lock step; a lane's extra candidates lie outside
                // its tile's support (weight exactly 0) or read the zero columns of the residual row
                if (ori == 0)      bs_walk<0>(rp, vp, n, 0, 0, true, xc0, yc0, sa.hka, sa.hkb, acc);
                else if (ori == 1) bs_walk<1>(rp, vp, n, 0, 0, true, xc0, yc0, sa.hka, sa.hkb, acc);
                else               bs_walk<2>(rp, vp, n, rel, (ori - 2) >> 1, (ori & 1) == 0, xc0, yc0, sa.hka, sa.hkb, acc);
                if (jl == ss && round == 0) OSIV_TL(a.iter, 1, 14, true);
            }
        }
    }
    OSIV_TL(a.iter, 1, 3, true);
    // A3 in the warp that leaves the walk first (it has the most slack before the block barrier): the
    // monitor partials in sum_partials' order (lane, lane + 32, ...), the step rule, the step for the epilogue
    if (MODE == 1) {
        int ticket = 0;
        if (lane == 0) ticket = atomicAdd(s_ticket, 1);
        ticket = __shfl_sync(0xffffffffu, ticket, 0);
        if (ticket == 0) {
            double dpv[BS_DPK];
#pragma unroll
            for (int k = 0; k < BS_DPK; ++k) dpv[k] = lane + 32 * k < a.nparts ? dp_s[lane + 32 * k] : 0.0;
            const SliceState st_in = *reinterpret_cast<const SliceState*>(st_s);
            double D = 0.0;
#pragma unroll
            for (int k = 0; k < BS_DPK; ++k) if (lane + 32 * k < a.nparts) D += dpv[k];
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) D += __shfl_xor_sync(0xffffffffu, D, off);
            const StepInfo si = step_decide(a, s, D, st_in, lane, b == 0);
            if (lane == 0) { s_step[0] = (float)(si.lambda * a.tau); reinterpret_cast<int*>(s_step)[1] = si.improved; }
        }
    }
    // the shares' sums meet in shared memory: red[(share q, tile i)][pixel p] = components 0..3 of the orbit's residuals
    {
        float4* rr = red + (size_t)(q * tpbp + i) * BS_RED_PITCH;
#pragma unroll
        for (int p = 0; p < BS_PX; ++p) {
            float c0, c1, c2, c3;
            unpack2(acc[0][p], c0, c1);
            unpack2(acc[1][p], c2, c3);
            rr[p] = make_float4(c0, c1, c2, c3);
        }
    }
    __syncthreads();
    OSIV_TL(a.iter, 1, 4, false);
    if (!fin) return;
    // share qq worked on quarter turn qq & 3: rotation k of the pixel collects component (k + quarter) & 3; fixed order
    float gsum[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int qq = 0; qq < BS_SHARES; ++qq) {
        const float4 v = red[(size_t)(qq * tpbp + ie) * BS_RED_PITCH + pe];
        const float c[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) gsum[k] += c[(k + qq) & 3];
    }
    const int rx[4] = {px, N - 1 - py, N - 1 - px, py}, ry[4] = {py, px, N - 1 - py, N - 1 - px};      // R^k P
    // padded offsets of R^k P in Q and of its transposed position in QT (square grid: one pitch): with A = (px+1) pitch,
    // B = (py+1) pitch and (N - x) pitch = (N+1) pitch - (x+1) pitch the eight offsets are sums of two products
    const int pA = (px + PADR) * g.pitch, pB = (py + PADR) * g.pitch, pN = (N - 1 + 2 * PADR) * g.pitch, n1 = N - 1;
    const int oq[4] = {pB + PAD + px, pA + PAD + n1 - py, pN - pB + PAD + n1 - px, pN - pA + PAD + py};
    const int ot[4] = {pA + PAD + py, pN - pB + PAD + px, pN - pA + PAD + n1 - py, pB + PAD + n1 - px};
    if constexpr (MODE == 0) {
        float* out = a.out + (size_t)s * N * N;
#pragma unroll
        for (int k = 0; k < 4; ++k) out[(size_t)ry[k] * N + rx[k]] = gsum[k];
    } else {
        // ---- A6 update (Eq. 3) with mu >= 0; the float4 of R^k P is the orbit read from k on
        const float step = s_step[0];
        float un[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) un[k] = fmaxf(fmaf(step, gsum[k] - a.beta_over_M * tv[k], cur[k]), 0.f);
        float4* Qn = reinterpret_cast<float4*>(a.img_new) + (size_t)s * g.img_elems;
        float4* QTn = reinterpret_cast<float4*>(a.imgT_new) + (size_t)s * g.imgT_elems;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const float4 v = make_float4(un[k], un[(k + 1) & 3], un[(k + 2) & 3], un[(k + 3) & 3]);
            Qn[oq[k]] = v;
            QTn[ot[k]] = v;
        }
        if (a.best && reinterpret_cast<const int*>(s_step)[1]) {             // A7: mu(n) had the smallest monitor so far
            float* best = a.best + (size_t)s * N * N;
#pragma unroll
            for (int k = 0; k < 4; ++k) best[(size_t)ry[k] * N + rx[k]] = cur[k];
        }
    }
    OSIV_TL(a.iter, 1, 5, true);
}

}  // namespace osiv
