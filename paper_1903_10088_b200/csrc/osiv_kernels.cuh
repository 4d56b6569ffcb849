// osiv_kernels.cuh -- sm_100a device code of libosiv (see include/osiv.h).
//
// Hot path of arxiv 1903.10088: per ordered-subset iteration
//   K1  k_forward<1,NS>  ray-driven reprojection l = A_S mu, fused Poisson residual and the per-ray-group
//                        fp64 partial sums of the monitor D
//   K2  k_back<1,NS>     monitor D (fixed-order sum of the partials) and the adaptive-step rule Eq. 4-5,
//                        matched atomic-free gather backprojection g = A_S^T r, fused TV gradient,
//                        Eq. 3 update, mu > 0 clamp, best-image copy; double-buffered image
//
// System matrix (reading C2): a(i,r) = length of the zero-width ray i inside square pixel r.  With
// p the signed distance of the pixel centre from the ray, the chord is the trapezoid
//   a = h * sat((hi - |p|) / (hi - lo)),  h = D/max(|dx|,|dy|), hi = D(|dx|+|dy|)/2, hi-lo = D*min(|dx|,|dy|).
// p is affine in the centred pixel indices (xc, yc), so after dividing by (hi-lo) every ray carries
// {alpha, beta, g0, h} (stored as the float4 {alpha, beta, g0, (|alpha|+|beta|)/2} plus a separate h table) with
//   a(i; xc,yc) = h * sat( (|alpha|+|beta|)/2 - |alpha*xc + beta*yc + g0| ),
// one of alpha,beta being exactly +-1 and the other |k| >= 1 (second model, Joseph's interpolation: the table holds
// the coefficients divided by |k| and a half-width of 1, a = h * sat(1 - |q|/|k|); the kernels do not change).
// Forward and back evaluate this same
// expression, so the pair is matched by construction.  Nothing here is a dense contraction: no
// tensor cores; the work is FP32 FMA/ALU issue plus L1/L2 gathers.
//
// Quarter-turn symmetry (NS = 4).  When the grid is square with nx % 4 == 0, V % 4 == 0 and the subset
// holds whole orbits {v, v+V/4, v+V/2, v+3V/4}, the scan is invariant under the rotation
// R: (xc,yc) -> (-yc,xc), i.e. pixel (ix,iy) -> (N-1-iy, ix):  a(v + kV/4, c; R^k P) = a(v, c; P).
// Every chord weight is then evaluated once and used for the four rotated (ray, pixel) pairs.  The image of this path
// is stored ORBIT-INTERLEAVED: one float4 per pixel P holding {mu(P), mu(RP), mu(R^2P), mu(R^3P)} (array Q, row-major,
// plus its transpose QT so that rays of either orientation walk contiguous lines), so K1 walks ray (v,c) with ONE
// 16-byte gather per touched pixel for all four rays of the orbit (the load/store unit issues one warp load per ~1.8
// cycles whatever its width, and the four scalar gathers of the earlier layout were K1's bound); K2 evaluates a(v,c;T)
// for its base tile T and feeds the accumulators of T, RT, R^2T, R^3T with the residuals of views v, v+V/4, v+V/2,
// v+3V/4, and its epilogue finishes one base pixel in all four rotations from the 3x3 neighbourhood of float4s.  The ray table is built with exactly
// rotated coefficients (alpha,beta,g0,h) -> (-beta,alpha,g0,h), so both kernels still use one weight per
// (ray, pixel) pair.  NS = 1 is the general path (any geometry).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace osiv {

// ---- phase timeline (diagnostics; only in the build with -DOSIV_TRACE, `python -m paper_1903_10088_b200.build --trace`):
// every block of the two hot kernels of slice group 0 stamps its SM's cycle counter (clock64: a few cycles per stamp) at
// its phase boundaries into g_timeline[(iteration & 1) * 2 + kernel][block][slot]; slots: 0 block start, 1 before the
// dependent-launch wait, 2 after it, 3 end of the main loop (latest warp), 4 after the block barrier, 5 block end (latest
// warp), 6 = SM id, 7 = a mark inside the prologue (K1: own ray loaded and clipped, before the first barrier; K2: tile
// origin known), 8 = %globaltimer [ns] read right after slot 0 (ties the SM's cycle counter to the device-wide clock).
constexpr int TL_BLOCKS = 256, TL_SLOTS = 16;
#ifdef OSIV_TRACE
__device__ unsigned long long g_timeline[4][TL_BLOCKS][TL_SLOTS];
__device__ __forceinline__ void tl_stamp(int iter, int kernel, int slot, bool latest) {
    if (blockIdx.z != 0 || blockIdx.x >= TL_BLOCKS) return;
    unsigned long long* row = g_timeline[(iter & 1) * 2 + kernel][blockIdx.x];
    if (latest) { if ((threadIdx.x & 31) == 0) atomicMax(&row[slot], (unsigned long long)clock64()); }
    else if (threadIdx.x == 0) {
        row[slot] = (unsigned long long)clock64();
        if (slot == 0) {
            unsigned sm; unsigned long long gt;
            asm volatile("mov.u32 %0, %%smid;" : "=r"(sm));
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt));
            row[6] = sm; row[8] = gt;
            row[3] = 0; row[5] = 0; for (int k = 9; k < TL_SLOTS; ++k) row[k] = 0;     // the "latest warp" slots restart for this launch
        }
    }
}
#define OSIV_TL(iter, kernel, slot, latest) tl_stamp(iter, kernel, slot, latest)
#else
#define OSIV_TL(iter, kernel, slot, latest) do {} while (0)
#endif

// ---- index checks (diagnostics; only in the build with -DOSIV_CHECKED, `python -m paper_1903_10088_b200.build --check`;
// compute-sanitizer is closed on the pool this was developed on): the gathers of both hot kernels rely on clamped indices
// landing in zero padding and on reads past a row's last channel staying inside the buffers; every such index is
// compared with its buffer's extent, g_check = {violations, site of the first one, checks made}.
#ifdef OSIV_CHECKED
__device__ unsigned long long g_check[4];
__device__ __forceinline__ void osiv_check(bool ok, int site) {
    if (!ok) { if (atomicAdd(&g_check[0], 1ull) == 0ull) g_check[1] = (unsigned long long)site; }
    else if ((threadIdx.x & 31) == 0) atomicAdd(&g_check[2], 1ull);
}
#define OSIV_CHECK(cond, site) osiv_check((cond), (site))
#else
#define OSIV_CHECK(cond, site) do {} while (0)
#endif

constexpr int PAD = 4;                     // zero columns left and right of every padded image line
constexpr int PADR = 1;                    // zero rows above and below a padded image
constexpr int FWD_MAX_THREADS = 1024;      // K1: one block per SM, threads = rays per block x line segments per ray
constexpr int FWD_MIN_LINES = 8;           // K1: a segment is at least this many image lines
constexpr int BK_TX = 2, BK_TY = 2;        // pixels per thread in the backprojector
constexpr int BK_WX = 8, BK_WY = 4;        // tiles per warp: a warp covers 16 x 8 pixels
constexpr int BKB_MAX_THREADS = 448;       // K2 serving two slices per block (SB == 2): two such blocks per SM
constexpr int BK_MAX_THREADS = 1024;       // K2: one block per SM, threads = tiles per block x view shares

struct DevGeom {
    int nx, ny, V, C;
    int pitch, pitchT;                     // floats per padded line of img ([ny+2][nx+8]) and imgT ([nx+2][ny+8])
    long long img_elems, imgT_elems;       // padded pixels per slice
    int sb;                                // slices interleaved per pixel in the padded images: 1, or 2 (launches with several slices)
    float cx, cy;                          // (nx-1)/2, (ny-1)/2
    float pixel, sad, inv_dgamma, c_center;   // c_center = (C-1)/2 - channel_offset
    float tile_hw;                         // angular half-width of a K2 tile at unit distance, in channels (with asin slack)
    int use_atanf;                         // fan too wide for the short atan polynomial
    int sym4;                              // geometry admits the quarter-turn path (square grid, nx%4==0, V%4==0)
    const float4* rays;                    // [V][C] {alpha, beta, g0, hk}, hk = (|alpha|+|beta|)/2 (both kernels' inner loops)
    const float* hs;                       // [V][C] chord scale h (per ray, outside the inner loops)
    const float2* views;                   // [V] {cos th_v, sin th_v}
};

struct SliceState {
    double lambda, D_prev, D_best, D_last;
    int n;                                 // subset updates done = next trace row
    int improved;                          // last monitor value beat D_best (return_best)
    int pad0, pad1;
};

struct IterParams {
    double lambda0, up, down, lmin;
    const double* forced;                  // device, [n_iters] or null
    double* trace;                         // device, [batch][n_iters][2] or null
    int n_iters;
    int return_best;
    int monitor_mode;                      // 0: compare with D(n-1); 1: with D(n-M) (same subset)
    int M;
    double* dhist;                         // monitor_mode 1: [batch][2M] ring of the last 2M monitor values
};

constexpr int FWD_ORDER_MAX = 160;         // K1 blocks per slice whose order travels in the kernel parameters

struct FwdArgs {
    DevGeom g;
    const float* img;                      // padded mu, slice stride g.img_elems
    const float* imgT;                     // padded transpose, slice stride g.imgT_elems
    int subset, M, VS;
    int batch;                             // slices in this launch (SB == 2: the last pair may be half empty)
    int view_shift;                        // stack of slices (H1): slice s uses the table's view (v + view_shift*s) mod V
    int rpb, segs;                         // rays per block, line segments per ray (block = rpb * segs threads, rounded up to warps)
    unsigned rpb_magic, C_magic;           // fastdiv by rpb and by g.C
    int iter;                              // iteration number (timeline build only)
    const int4* rng_tab;                   // [M][gridDim.x] line ranges of every block's row- / column-major rays {lo, hi, lo, hi}
                                           // (k_build_fwd_ranges), or null: the block works them out itself (stacks)
    const float* invk;                     // [V][C] 1 / (in-line coefficient) of every ray, or null
    unsigned segs_magic;
    float* sino;                           // MODE 0: [batch][VS][C]
    const float* counts;                   // MODE 1: [batch][V][C]
    const float* blank;                    // [C] or null
    float blank_scalar;
    const float* inv_bref;                 // device scalar 1/b_ref
    float* res;                            // MODE 1: h * r; NS == 1: [batch][VS][Cp] floats, NS == 4: [batch][VS/4][Cp] float4
                                           // holding the orbit {j, j+VS/4, j+VS/2, j+3VS/4}; columns C..Cp-1 stay zero
    int Cp;
    double* dparts;                        // MODE 1: [batch][gridDim.x] partial sums of D
    long long res_floats;                  // floats in `res` (checked build)
    // Blocks are handed to the SMs in blockIdx order as the predecessor's blocks exit, about a microsecond between the
    // first and the last: order[blockIdx.x] = the run of rays this block takes, the runs with the longest walks first
    // (from the tabulated line ranges, per subset), so that the late starters are the short ones.  In the kernel
    // parameters (constant bank): a table in memory would put a round trip at the head of the start-up path.
    int use_order;
    unsigned short order[FWD_ORDER_MAX];
};

struct BackArgs {
    DevGeom g;
    const float* res;                      // h * (residual or sinogram), layout as FwdArgs::res
    int Cp;
    int subset, M, VS;
    int batch;                             // slices in this launch (SB == 2: the last pair may be half empty)
    int view_shift;                        // stack of slices (H1), as in FwdArgs
    float tv_z;                            // stack of slices (H2): > 0 adds the z term of the 3-D TV (SB == 1 only)
    int tpb, shares, ngx;                  // tiles per block, view shares, 2x2 patch groups per row of groups
    unsigned tpb_magic, ngx_magic;         // fastdiv by tpb and by ngx
    int iter;                              // iteration number (timeline build only)
    const int* itab;                       // [V][ntiles] candidate intervals (k_build_intervals)
    int ntiles;
    float* out;                            // MODE 0: [batch][ny][nx]
    const float* img;                      // MODE 1: padded mu(n)
    float* img_new;                        // padded mu(n+1)
    float* imgT_new;
    float* best;                           // [batch][ny][nx] or null
    const double* dparts;                  // [batch][nparts]
    int nparts;
    const SliceState* state_in;            // [batch] state after iteration n-1
    SliceState* state_out;                 // [batch] state after iteration n
    int* not_finite;                       // [batch] sticky flags
    IterParams ip;
    double tau;
    float beta_over_M, eps2;
    long long res_floats, ray_entries;     // floats in `res`, float4 entries behind g.rays (checked build)
};

// n / d for 0 <= n < 2^32 / d with the host's magic = ceil(2^32 / d) (0 for d = 1): one multiply instead of the division
// sequence (the start-up path of both hot kernels lies on the iteration's critical path)
__device__ __forceinline__ int fastdiv(int n, unsigned magic) { return magic ? (int)__umulhi((unsigned)n, magic) : n; }

__device__ __forceinline__ size_t pad_off(const DevGeom& g, int iy, int ix) {
    return (size_t)(iy + PADR) * g.pitch + PAD + ix;
}
__device__ __forceinline__ size_t padT_off(const DevGeom& g, int ix, int iy) {
    return (size_t)(ix + PADR) * g.pitchT + PAD + iy;
}
// float index of padded pixel 0 of slice s: slices are stored in groups of g.sb, interleaved per pixel, so pixel p of
// slice s lives at slice_base + p * g.sb
__device__ __forceinline__ size_t slice_base(const DevGeom& g, long long elems, int s) {
    return (size_t)(s / g.sb) * (size_t)elems * g.sb + (size_t)(s % g.sb);
}

// ---- programmatic dependent launch: both hot kernels are launched while their predecessor in the stream still runs;
// everything above pdl_wait() touches only constants (geometry tables, indices), pdl_wait() returns once the
// predecessor has completed and its writes are visible, and pdl_launch_next() -- placed AFTER the wait, so that at
// most one successor is ever resident early -- lets the successor's blocks move into the SM slots this grid frees.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
// Pins a value of the prologue in front of the wait.  ptxas treats griddepcontrol.wait (ACQBULK) like a long-latency
// operation and hoists it to the top of its basic block -- above the constant-memory loads and the arithmetic of a
// straight-line prologue, which then runs only after the predecessor has completed (seen in the SASS); it does not move
// it across a warp barrier, so the value is made an operand of one.
__device__ __forceinline__ void pdl_before_wait(int x) { asm volatile("bar.warp.sync 0xffffffff;" ::"r"(x) : "memory"); }
__device__ __forceinline__ void pdl_launch_next() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// Packed FP32 pairs (Blackwell FFMA2: two IEEE fp32 FMAs per instruction, the scalar operand broadcast): halves the
// issue slots of the accumulation, bit-identical to two FFMAs.
__device__ __forceinline__ uint64_t pack2(float lo, float hi) {
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(uint64_t v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ void ffma2(uint64_t& c, uint64_t a, float b) {       // c += a * (b, b)
    const uint64_t bb = pack2(b, b);
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(c) : "l"(a), "l"(bb));
}

// ------------------------------------------------------------------------------------------------
// K1: forward projection (+ residual and monitor partials when MODE == 1).
// One block per SM-sized share of the subset's base rays: the R = (V_S/NS) * C base rays are dealt out in runs of
// `rpb` consecutive rays (view-major), and a block is rpb rays x `segs` segments of each ray's own image-line range
// [flo, fhi]: thread t walks segment t / rpb of ray t % rpb.  Neighbouring threads are neighbouring channels on
// the same line (the block walks the union of its rays' ranges in lock step), so a warp's gathers fall into one or two cache lines.  A ray marches over the image lines
// of its major axis (rows of img when |dy| >= |dx|, else rows of the transposed copy imgT) and touches at most two
// adjacent pixels per line; with NS == 4 the same two weights also serve the three rotated rays.  Every block has
// the same amount of work and no block depends on another: the segment sums meet in shared memory in a fixed order
// and the first rpb threads run the per-ray epilogue.  The host sizes the grid to one block per SM (fwd_plan).
// ------------------------------------------------------------------------------------------------
// SB == 2 (launches with several slices, A8): a block serves a pair of slices whose padded images are interleaved per
// pixel (DevGeom::sb == 2), so every gather is one float2 = the pixel in both slices, the chord weights -- the bulk of
// K1's instructions -- are worked out once per pair, and the FFMA2 pairs run over the two slices.
// image lines [flo, fhi] of the ray's major axis on which its crossing lies within half a pixel of the image:
// |uu*b + g0| < |kk|*(na/2 + 1/2)
__device__ __forceinline__ void ray_lines(const DevGeom& g, const float4 ray, int& flo, int& fhi) {
    const bool rowmaj = fabsf(ray.x) >= fabsf(ray.y);
    const float kk = rowmaj ? ray.x : ray.y, uu = rowmaj ? ray.y : ray.x;
    const int na = rowmaj ? g.nx : g.ny, nb = rowmaj ? g.ny : g.nx;
    const float cb = rowmaj ? g.cy : g.cx;
    const float A = fabsf(kk) * (0.5f * na + 0.5f);
    const float iu = 1.0f / uu;                           // exact chord: uu = +-1; Joseph: |uu| <= 1
    const float b1 = iu * (-ray.z - A), b2 = iu * (-ray.z + A);
    flo = (int)fminf(fmaxf(ceilf(fminf(b1, b2) + cb) - 1.f, 0.f), (float)nb);
    fhi = (int)fminf(fmaxf(floorf(fmaxf(b1, b2) + cb) + 1.f, -1.f), (float)(nb - 1));
}

// A0 for K1, once per handle, subset count and block shape: the union of line ranges of every block's row-major and
// column-major rays (what k_forward otherwise works out with two block barriers at every launch).  grid (blocks, M).
__global__ void __launch_bounds__(1024) k_build_fwd_ranges(DevGeom g, int M, int VS, int ns, int rpb, int4* __restrict__ tab) {
    __shared__ int rng[4];
    const int i = threadIdx.x, m = blockIdx.y;
    if (i < 4) rng[i] = (i & 1) ? -1 : (1 << 30);
    __syncthreads();
    const int VSb = VS / ns, R = VSb * g.C, r = blockIdx.x * rpb + i;
    if (i < rpb && r < R) {
        const int jb = r / g.C, c = r - jb * g.C;
        const int v = m + jb * M;
        const float4 ray = __ldg(&g.rays[(size_t)v * g.C + c]);
        int flo, fhi;
        ray_lines(g, ray, flo, fhi);
        if (fhi >= flo) {
            const int o = fabsf(ray.x) >= fabsf(ray.y) ? 0 : 2;
            atomicMin(&rng[o], flo); atomicMax(&rng[o + 1], fhi);
        }
    }
    __syncthreads();
    if (i == 0) tab[(size_t)m * gridDim.x + blockIdx.x] = make_int4(rng[0], rng[1], rng[2], rng[3]);
}

template <int SB> struct Px;
template <> struct Px<1> { typedef float T; };
template <> struct Px<2> { typedef float2 T; };

template <int MODE, int NS, int SB>
__global__ void __launch_bounds__(FWD_MAX_THREADS, 1) k_forward(const FwdArgs a) {
    typedef typename Px<SB>::T PX;
    const DevGeom& g = a.g;
    const int t = threadIdx.x, s0 = blockIdx.z * SB;             // slices s0 .. s0 + SB - 1
    OSIV_TL(a.iter, 0, 0, false);
    const int rpb = a.rpb, segs = a.segs;
    const int seg = fastdiv(t, a.rpb_magic), i = t - seg * rpb;
    const int VSb = a.VS / NS, Vq = g.V / NS;
    const int R = VSb * g.C;
    const int bx = a.use_order ? (int)a.order[blockIdx.x] : (int)blockIdx.x;      // the run of rays of this block
    const int r = bx * rpb + i;
    const bool walker = seg < segs && r < R;
    const int rr = min(r, R - 1);
    const int jb = fastdiv(rr, a.C_magic), c = rr - jb * g.C;
    const int v = a.subset < 0 ? jb : a.subset + jb * a.M;          // base view of the orbit
    extern __shared__ float part[];                                 // [segs][NS][SB][rpb]
    __shared__ double dred[2][FWD_MAX_THREADS / 32];
    __shared__ int rng[4];                                          // line ranges of the block's row- / column-major rays

    float acc[1] = {0.f};                                           // NS == 1, SB == 1
    uint64_t acc2[1] = {0ull};                                      // NS == 1, SB == 2: the pair of slices
    uint64_t acc4[SB][2];                                           // NS == 4: per slice, orbit rays (0, 1) and (2, 3)
#pragma unroll
    for (int sl = 0; sl < SB; ++sl) { acc4[sl][0] = 0ull; acc4[sl][1] = 0ull; }
    // H1: a slice of a stack sees the gantry view_shift views further on per slice; the counts keep the acquisition index
    int vt = v;                                                     // (a real branch: the default path must not pay for the modulo)
    if (a.view_shift) { vt = v + (int)(((unsigned)a.view_shift * (unsigned)s0) % (unsigned)g.V); if (vt >= g.V) vt -= g.V; }
    const float4 ray = __ldg(&g.rays[(size_t)vt * g.C + c]);
    const bool rowmaj = fabsf(ray.x) >= fabsf(ray.y);
    {
        const float kk = rowmaj ? ray.x : ray.y;          // coefficient of the in-line coordinate, |kk| >= 1 (Joseph: +-1)
        const float uu = rowmaj ? ray.y : ray.x;          // coefficient of the marching coordinate (+-1; Joseph: +-1/|k|)
        const PX* bufA = rowmaj ? reinterpret_cast<const PX*>(a.img) + (size_t)blockIdx.z * g.img_elems : reinterpret_cast<const PX*>(a.imgT) + (size_t)blockIdx.z * g.imgT_elems;
        // NS == 4: the orbit-interleaved image Q (rays crossing rows) or its transpose QT (rays crossing columns), SB float4 per pixel
        // (slice-major, NOT interleaved per pixel: with two slices' float4s side by side a warp's 16-byte gathers are strided by 32
        // bytes and every L1 wavefront carries half its width -- 12.9 k instead of 8.5 k wavefronts per slice and SM, ncu)
        const long long q_plane = rowmaj ? g.img_elems : g.imgT_elems;
        const float4* qA = reinterpret_cast<const float4*>(rowmaj ? a.img : a.imgT) + (size_t)blockIdx.z * q_plane * SB;
        const int pitch = rowmaj ? g.pitch : g.pitchT;    // NS == 4: square grid, both pitches are equal
        const int na = rowmaj ? g.nx : g.ny;
        const float ca = rowmaj ? g.cx : g.cy, cb = rowmaj ? g.cy : g.cx;
        const float invk = a.invk ? __ldg(&a.invk[(size_t)vt * g.C + c]) : 1.0f / kk;
        const float hk = ray.w;
        // The block walks the union of its rays' line ranges in lock step, so that at every step the lanes of a warp
        // read neighbouring pixels of ONE image line (1-2 cache lines per load instead of up to 32; rays clipped by an
        // image corner start many lines apart).  On a line outside a ray's own range the crossing is more than half a
        // pixel outside the image: the clamped index lands in the zero padding and the term vanishes.
        // (Row-major and column-major rays of one block form two such unions: their lines are different things.)
        int wlo, whi;
        OSIV_TL(a.iter, 0, 7, false);
        if (a.rng_tab) {                                      // tabulated (A0): no barrier in the start-up path
            const int4 rg = __ldg(&a.rng_tab[(size_t)(a.subset < 0 ? 0 : a.subset) * gridDim.x + bx]);
            wlo = rowmaj ? rg.x : rg.z; whi = rowmaj ? rg.y : rg.w;
        } else {
        int flo, fhi;
        ray_lines(g, ray, flo, fhi);
        if (t < 4) rng[t] = (t & 1) ? -1 : (1 << 30);
        __syncthreads();
        {
            const int big = 1 << 30;
            const int lo = __reduce_min_sync(0xffffffffu, walker && rowmaj ? flo : big);
            const int hi = __reduce_max_sync(0xffffffffu, walker && rowmaj ? fhi : -1);
            const int lo2 = __reduce_min_sync(0xffffffffu, walker && !rowmaj ? flo : big);
            const int hi2 = __reduce_max_sync(0xffffffffu, walker && !rowmaj ? fhi : -1);
            if ((t & 31) == 0) {
                if (hi >= lo) { atomicMin(&rng[0], lo); atomicMax(&rng[1], hi); }
                if (hi2 >= lo2) { atomicMin(&rng[2], lo2); atomicMax(&rng[3], hi2); }
            }
        }
        __syncthreads();
        wlo = rowmaj ? rng[0] : rng[2]; whi = rowmaj ? rng[1] : rng[3];
        }
        const int nsteps = walker ? max(whi - wlo + 1, 0) : 0;
        const int len = fastdiv(nsteps + segs - 1, a.segs_magic);
        const int j0 = wlo + seg * len;
        const int j1 = min(j0 + len, wlo + nsteps);
        const int imax = na + PAD - 2;
        int offP = (j0 + PADR) * pitch + PAD;                 // line j, walking up
        float bf = (float)j0 - cb;
        OSIV_TL(a.iter, 0, 1, false);
        pdl_wait();                                           // mu(n) is the previous launch's output
        pdl_launch_next();
        OSIV_TL(a.iter, 0, 2, false);
        // LPT lines per trip, written so that all gathers of a trip are in flight together: the walk is bound by the
        // load path.  The lines past j1 (only in the last trip) get zero weights; with two lines per trip their addresses
        // stay inside the padded buffers because j1 <= nb, with more the last valid line is read again.
        // floor() by the add-a-big-number trick (|t| < 2^22; FRND/F2I run at a quarter of the FP32 rate): r = t - 1/2 +
        // 1.5 * 2^23 rounds to the nearest integer, which is floor(t) unless t is an integer n, where it may be n - 1:
        // then pixels n - 1 and n are taken instead of n and n + 1, and both left-out pixels are a whole pixel away
        // from the crossing (weight 0 in either model).
        constexpr float BIG = 12582912.f;
        // image lines per trip: four on the one-slice quarter-turn path (eight 16-byte gathers in flight per thread; A/B at
        // config 3: 2 lines 56.5 k, 3 55.9 k, 4 57.0 k, 5 55.8 k, 6 55.7 k, 7 56.4 k iterations/s), two elsewhere
        constexpr int LPT = (NS == 4 && SB == 1) ? 4 : 2;
        for (int jj = j0; jj < j1; jj += LPT, offP += LPT * pitch, bf += (float)LPT) {
            float w[LPT][2];
            int i0[LPT];
#pragma unroll
            for (int u = 0; u < LPT; ++u) {
                const float bg = fmaf(uu, bf + (float)u, ray.z);
                const float r = (fmaf(-bg, invk, ca) - 0.5f) + BIG;
                const float fa = r - BIG;                         // index of the pixel left of the crossing
                const float q0 = fmaf(kk, fa - ca, bg);
                const float q1 = q0 + kk;
                w[u][0] = __saturatef(hk - fabsf(q0));
                w[u][1] = __saturatef(hk - fabsf(q1));
                i0[u] = min(max(__float_as_int(r) - 0x4B400000, -PAD), imax);
            }
#pragma unroll
            for (int u = 1; u < LPT; ++u)
                if (jj + u >= j1) { w[u][0] = 0.f; w[u][1] = 0.f; }
            if constexpr (NS == 4) {
                // one float4 per pixel and slice = the pixel in the four rotated positions: component k belongs to ray
                // (v + k V/4, c) of the orbit, with the same weight
                float4 x[LPT][2][SB];
#pragma unroll
                for (int u = 0; u < LPT; ++u) {
                    const int ul = LPT > 2 ? min(u, j1 - jj) : u;      // lines past the segment's end: any valid line (weights 0)
                    OSIV_CHECK(offP + ul * pitch + i0[u] >= 0 && offP + ul * pitch + i0[u] + 1 < (rowmaj ? g.img_elems : g.imgT_elems), 1);
                    const float4* p0 = qA + (offP + ul * pitch + i0[u]);
#pragma unroll
                    for (int e = 0; e < 2; ++e)
#pragma unroll
                        for (int sl = 0; sl < SB; ++sl) x[u][e][sl] = __ldg(p0 + sl * q_plane + e);
                }
#pragma unroll
                for (int u = 0; u < LPT; ++u)
#pragma unroll
                    for (int e = 0; e < 2; ++e)
#pragma unroll
                        for (int sl = 0; sl < SB; ++sl) {
                            ffma2(acc4[sl][0], pack2(x[u][e][sl].x, x[u][e][sl].y), w[u][e]);
                            ffma2(acc4[sl][1], pack2(x[u][e][sl].z, x[u][e][sl].w), w[u][e]);
                        }
            } else {
                PX x[2][2];
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    OSIV_CHECK(offP + u * pitch + i0[u] >= 0 && offP + u * pitch + i0[u] + 1 < (rowmaj ? g.img_elems : g.imgT_elems), 2);
                    const PX* p0 = bufA + (offP + u * pitch + i0[u]);
                    x[u][0] = __ldg(p0); x[u][1] = __ldg(p0 + 1);
                }
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    if constexpr (SB == 2) {                      // the two slices as an FFMA2 pair
                        ffma2(acc2[0], pack2(x[u][0].x, x[u][0].y), w[u][0]);
                        ffma2(acc2[0], pack2(x[u][1].x, x[u][1].y), w[u][1]);
                    } else {
                        acc[0] = fmaf(w[u][0], x[u][0], acc[0]);
                        acc[0] = fmaf(w[u][1], x[u][1], acc[0]);
                    }
                }
            }
        }
    }
    OSIV_TL(a.iter, 0, 3, true);
    // this thread's sums: fin[ray of the orbit][slice of the block]
    float fin[NS][SB];
    if constexpr (NS == 4) {
#pragma unroll
        for (int sl = 0; sl < SB; ++sl) {
            unpack2(acc4[sl][0], fin[0][sl], fin[1 % NS][sl]);
            unpack2(acc4[sl][1], fin[2 % NS][sl], fin[3 % NS][sl]);
        }
    } else if constexpr (SB == 2) {
        unpack2(acc2[0], fin[0][0], fin[0][SB - 1]);
    } else {
        fin[0][0] = acc[0];
    }
    if (seg < segs) {
#pragma unroll
        for (int k = 0; k < NS; ++k)
#pragma unroll
            for (int sl = 0; sl < SB; ++sl) part[((seg * NS + k) * SB + sl) * rpb + i] = fin[k][sl];
    }
    // Epilogue: thread (seg = ko < NS, ray i) finishes ray i of rotation ko -- its own ray, so everything about the ray
    // is in registers already.  Its inputs are requested before the barrier so that they arrive while the block drains.
    const int ne = min(segs, NS);                             // epilogue threads per ray
    const bool epi = seg < ne && r < R;
    float y0 = 0.f, bl = a.blank_scalar, ib = 0.f, h = 0.f;
    if (epi) h = __ldg(&g.hs[(size_t)vt * g.C + c]);
    if (MODE == 1 && epi) {
        y0 = __ldg(&a.counts[((size_t)s0 * g.V + v + seg * Vq) * g.C + c]);
        if (a.blank) bl = __ldg(&a.blank[c]);
        ib = __ldg(a.inv_bref);
    }
    __syncthreads();
    OSIV_TL(a.iter, 0, 4, false);
    const int nw = (ne * rpb + 31) / 32;                      // epilogue warps
    if (t >= 32 * nw) return;

    double d2[SB];
#pragma unroll
    for (int sl = 0; sl < SB; ++sl) d2[sl] = 0.0;
    if (epi) {
        for (int ko = seg; ko < NS; ko += ne) {
            const int pk = ko;
#pragma unroll
            for (int sl = 0; sl < SB; ++sl) {
                const int s = s0 + sl;
                if (s >= a.batch) break;
                // sum over the ray's segments in a fixed order: four interleaved partial sums, so that the loads do not
                // wait for one another
                float xs[4] = {0.f, 0.f, 0.f, 0.f};
                const float* pp = part + (pk * SB + sl) * rpb + i;
                const int stride = NS * SB * rpb;
                int q = 0;
                for (; q + 4 <= segs; q += 4) {
#pragma unroll
                    for (int e = 0; e < 4; ++e) xs[e] += pp[(q + e) * stride];
                }
                for (; q < segs; ++q) xs[0] += pp[q * stride];
                const float l = h * ((xs[0] + xs[1]) + (xs[2] + xs[3]));
                if (MODE == 0) {
                    a.sino[((size_t)s * a.VS + jb + ko * VSb) * g.C + c] = l;
                } else {
                    // A2: Poisson residual r = (b exp(-l) - y)/b_ref and monitor term (l - ln(b/max(y,1)))^2
                    const float y = (ko == seg && sl == 0) ? y0 : __ldg(&a.counts[((size_t)s * g.V + v + ko * Vq) * g.C + c]);
                    const float ybar = bl * expf(-l);
                    const float hr = h * ((ybar - y) * ib);
                    const float p = logf(bl / fmaxf(y, 1.f));
                    const double d = (double)l - (double)p;
                    d2[sl] += d * d;
                    // NS == 4: the orbit's four residuals share one float4 (K2 reads them with one load per candidate ray)
                    OSIV_CHECK((long long)((((size_t)s * VSb + jb) * a.Cp + c) * NS + ko) < a.res_floats, 3);
                    a.res[(((size_t)s * VSb + jb) * a.Cp + c) * NS + ko] = hr;
                }
            }
        }
    }
    if (MODE == 1) {
        // block's share of each slice's D: warp shuffles, then the (at most 32) warp sums in a fixed order
#pragma unroll
        for (int sl = 0; sl < SB; ++sl) {
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) d2[sl] += __shfl_down_sync(0xffffffffu, d2[sl], off);
            if ((t & 31) == 0) dred[sl][t >> 5] = d2[sl];
        }
        asm volatile("bar.sync 1, %0;" ::"r"(32 * nw) : "memory");     // only the epilogue warps meet here
        if (t < SB) {                                                  // one thread per slice: the warp sums in a fixed order
            double D = 0.0;
            for (int w = 0; w < nw; ++w) D += dred[t][w];
            if (s0 + t < a.batch) a.dparts[(size_t)(s0 + t) * gridDim.x + bx] = D;
        }
    }
    OSIV_TL(a.iter, 0, 5, true);
}

// ------------------------------------------------------------------------------------------------
// Monitor D(n) = fixed-order sum of K1's partials (every caller warp computes the same bits), then A3
// (Eq. 4-5).  Returns lambda(n) and whether D(n) beat D_best; `writer` publishes the state.
// ------------------------------------------------------------------------------------------------
struct StepInfo { double lambda; double D; int improved; };

__device__ __forceinline__ double sum_partials(const double* p, int n, int lane) {
    double D = 0.0;
    // lane l adds p[l], p[l + 32], ... in that order; eight loads in flight (a slot past the end adds an exact 0)
    for (int i0 = 0; i0 < n; i0 += 256) {
        double v[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) v[k] = i0 + lane + 32 * k < n ? __ldg(&p[i0 + lane + 32 * k]) : 0.0;
#pragma unroll
        for (int k = 0; k < 8; ++k) D += v[k];
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) D += __shfl_xor_sync(0xffffffffu, D, off);
    return D;
}

// A3 from the monitor value D(n) and the state after iteration n-1 (every lane of the calling warp holds both)
__device__ __forceinline__ StepInfo step_decide(const BackArgs& a, int s, double D, const SliceState& st, int lane, bool writer) {
    StepInfo si;
    si.D = D;
    const int n = st.n;
    double lam;
    if (a.ip.forced)          lam = a.ip.forced[n];
    else if (n < (a.ip.monitor_mode ? a.ip.M : 1)) lam = a.ip.lambda0;
    else if (si.D < (a.ip.monitor_mode ? a.ip.dhist[(size_t)s * 2 * a.ip.M + (n - a.ip.M) % (2 * a.ip.M)] : st.D_prev)) lam = st.lambda + a.ip.up;
    else                      lam = fmax(st.lambda - a.ip.down, a.ip.lmin);
    si.lambda = lam;
    si.improved = a.ip.return_best && si.D < st.D_best;
    if (writer && lane == 0) {
        SliceState o;
        o.lambda = lam; o.D_prev = si.D; o.D_best = si.improved ? si.D : st.D_best; o.D_last = si.D;
        o.n = n + 1; o.improved = si.improved; o.pad0 = 0; o.pad1 = 0;
        a.state_out[s] = o;
        if (!isfinite(si.D)) a.not_finite[s] = 1;
        // slot n % 2M is written while every block may still read slot (n - M) % 2M: never the same slot
        if (a.ip.monitor_mode) a.ip.dhist[(size_t)s * 2 * a.ip.M + n % (2 * a.ip.M)] = si.D;
        if (a.ip.trace) {
            double* tr = a.ip.trace + ((size_t)s * a.ip.n_iters + n) * 2;
            tr[0] = si.D;
            tr[1] = lam;
        }
    }
    return si;
}

__device__ __forceinline__ StepInfo step_rule(const BackArgs& a, int s, int lane, bool writer) {
    const double D = sum_partials(a.dparts + (size_t)s * a.nparts, a.nparts, lane);
    const SliceState st = a.state_in[s];
    return step_decide(a, s, D, st, lane, writer);
}

// final iterate's monitor (return_best): one warp per slice
__global__ void k_final_monitor(const double* dparts, int nparts, SliceState* state, int* not_finite) {
    const int s = blockIdx.x, lane = threadIdx.x;
    const double D = sum_partials(dparts + (size_t)s * nparts, nparts, lane);
    if (lane == 0) {
        state[s].D_last = D;
        state[s].improved = D < state[s].D_best;
        if (!isfinite(D)) not_finite[s] = 1;
    }
}

// ------------------------------------------------------------------------------------------------
// Smoothed isotropic TV gradient (reading C8) of the 2x2 tile whose 4x4 neighbourhood is m:
//   m[r][c] = mu(y0-1+r, x0-1+c).  Differences across the image border are 0, terms whose
// neighbour is outside are dropped.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void tv_grad_tile(const float (&m)[4][4], int x0, int y0, int nx, int ny,
                                             float eps2, float (&out)[2][2]) {
    // it[r][c] = 1/t at (y0-1+r, x0-1+c) for r,c in 0..2
    float it[3][3];
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const int x = x0 - 1 + c, y = y0 - 1 + r;
            const float dxv = (x + 1 < nx) ? m[r][c + 1] - m[r][c] : 0.f;
            const float dyv = (y + 1 < ny) ? m[r + 1][c] - m[r][c] : 0.f;
            it[r][c] = rsqrtf(eps2 + dxv * dxv + dyv * dyv);
        }
#pragma unroll
    for (int ty = 0; ty < 2; ++ty)
#pragma unroll
        for (int tx = 0; tx < 2; ++tx) {
            const int x = x0 + tx, y = y0 + ty, r = ty + 1, c = tx + 1;
            const float cv = m[r][c];
            float sgrad = 0.f;
            if (x > 0) sgrad += (cv - m[r][c - 1]) * it[r][c - 1];
            if (y > 0) sgrad += (cv - m[r - 1][c]) * it[r - 1][c];
            const float dxv = (x + 1 < nx) ? m[r][c + 1] - cv : 0.f;
            const float dyv = (y + 1 < ny) ? m[r + 1][c] - cv : 0.f;
            sgrad -= (dxv + dyv) * it[r][c];
            out[ty][tx] = sgrad;
        }
}

// The same with the z term of the 3-D TV (reading H2): up / dn = the neighbourhood in slices s+1 / s-1, wz = tv_z.
// Own cell: -(dx + dy + wz*Dz)/t with Dz = wz*(up - mu); cell below: +wz*Dz'/t' with Dz' = wz*(mu - dn).
__device__ __forceinline__ void tv_grad_tile3(const float (&m)[4][4], const float (&up)[4][4], const float (&dn)[4][4],
                                              bool has_up, bool has_dn, float wz, int x0, int y0, int nx, int ny,
                                              float eps2, float (&out)[2][2]) {
    float it[3][3];
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const int x = x0 - 1 + c, y = y0 - 1 + r;
            const float dxv = (x + 1 < nx) ? m[r][c + 1] - m[r][c] : 0.f;
            const float dyv = (y + 1 < ny) ? m[r + 1][c] - m[r][c] : 0.f;
            const float dzv = has_up ? wz * (up[r][c] - m[r][c]) : 0.f;
            it[r][c] = rsqrtf(eps2 + dxv * dxv + dyv * dyv + dzv * dzv);
        }
#pragma unroll
    for (int ty = 0; ty < 2; ++ty)
#pragma unroll
        for (int tx = 0; tx < 2; ++tx) {
            const int x = x0 + tx, y = y0 + ty, r = ty + 1, c = tx + 1;
            const float cv = m[r][c];
            float sgrad = 0.f;
            if (x > 0) sgrad += (cv - m[r][c - 1]) * it[r][c - 1];
            if (y > 0) sgrad += (cv - m[r - 1][c]) * it[r - 1][c];
            if (has_dn) {
                const float dxd = (x + 1 < nx) ? dn[r][c + 1] - dn[r][c] : 0.f;
                const float dyd = (y + 1 < ny) ? dn[r + 1][c] - dn[r][c] : 0.f;
                const float dzd = wz * (cv - dn[r][c]);
                sgrad += wz * dzd * rsqrtf(eps2 + dxd * dxd + dyd * dyd + dzd * dzd);
            }
            const float dxv = (x + 1 < nx) ? m[r][c + 1] - cv : 0.f;
            const float dyv = (y + 1 < ny) ? m[r + 1][c] - cv : 0.f;
            const float dzv = has_up ? wz * (up[r][c] - cv) : 0.f;
            sgrad -= (dxv + dyv + wz * dzv) * it[r][c];
            out[ty][tx] = sgrad;
        }
}

// Quarter-turn path: value and TV gradient (C8) of pixel R^K P from the 3x3 neighbourhood E of orbit float4s around the
// base pixel P = (px, py):  E[1+dy][1+dx] = {mu(P'), mu(RP'), mu(R^2P'), mu(R^3P')}, P' = P + (dx, dy).  The neighbour of
// R^K P at image offset (a, b) is R^K (P + R^-K (a, b)), i.e. component K of the entry at base offset R^-K (a, b).
template <int K> __device__ __forceinline__ float orbit_comp(const float4& v) { return K == 0 ? v.x : K == 1 ? v.y : K == 2 ? v.z : v.w; }
template <int K> __device__ __forceinline__ float orbit_nb(const float4 (&E)[3][3], int a, int b) {
    const int dx = K == 0 ? a : K == 1 ? b : K == 2 ? -a : -b;
    const int dy = K == 0 ? b : K == 1 ? -a : K == 2 ? -b : a;
    return orbit_comp<K>(E[1 + dy][1 + dx]);
}
// 1/sqrt(x) for x >= eps^2 > 0: the bare MUFU.RSQ (rsqrtf adds two scalings for denormal inputs that cannot occur here)
__device__ __forceinline__ float rsqrt_fast(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
template <int K>
__device__ __forceinline__ void orbit_tv(const float4 (&E)[3][3], int px, int py, int N, float eps2, float& cur, float& grad) {
    const int x = K == 0 ? px : K == 1 ? N - 1 - py : K == 2 ? N - 1 - px : py;        // R^K P
    const int y = K == 0 ? py : K == 1 ? px : K == 2 ? N - 1 - py : N - 1 - px;
    const bool hx1 = x + 1 < N, hy1 = y + 1 < N;
    const float c = orbit_nb<K>(E, 0, 0);
    const float dxc = hx1 ? orbit_nb<K>(E, 1, 0) - c : 0.f, dyc = hy1 ? orbit_nb<K>(E, 0, 1) - c : 0.f;
    float sgrad = 0.f;
    if (x > 0) {                                                     // cell (x-1, y)
        const float l = orbit_nb<K>(E, -1, 0), dxl = c - l, dyl = hy1 ? orbit_nb<K>(E, -1, 1) - l : 0.f;
        sgrad += dxl * rsqrt_fast(eps2 + dxl * dxl + dyl * dyl);
    }
    if (y > 0) {                                                     // cell (x, y-1)
        const float d = orbit_nb<K>(E, 0, -1), dyb = c - d, dxb = hx1 ? orbit_nb<K>(E, 1, -1) - d : 0.f;
        sgrad += dyb * rsqrt_fast(eps2 + dxb * dxb + dyb * dyb);
    }
    sgrad -= (dxc + dyc) * rsqrt_fast(eps2 + dxc * dxc + dyc * dyc);
    cur = c;
    grad = sgrad;
}

// The same for a pixel orbit off the image border (0 < px, py < N - 1; a quarter turn about the centre maps the border
// ring onto itself, so one test serves the four rotations): no predicates, the same float operations in the same order.
template <int K>
__device__ __forceinline__ void orbit_tv_inner(const float4 (&E)[3][3], float eps2, float& cur, float& grad) {
    const float c = orbit_nb<K>(E, 0, 0);
    const float dxc = orbit_nb<K>(E, 1, 0) - c, dyc = orbit_nb<K>(E, 0, 1) - c;
    float sgrad = 0.f;
    {                                                                // cell (x-1, y)
        const float l = orbit_nb<K>(E, -1, 0), dxl = c - l, dyl = orbit_nb<K>(E, -1, 1) - l;
        sgrad += dxl * rsqrt_fast(eps2 + dxl * dxl + dyl * dyl);
    }
    {                                                                // cell (x, y-1)
        const float d = orbit_nb<K>(E, 0, -1), dyb = c - d, dxb = orbit_nb<K>(E, 1, -1) - d;
        sgrad += dyb * rsqrt_fast(eps2 + dxb * dxb + dyb * dyb);
    }
    sgrad -= (dxc + dyc) * rsqrt_fast(eps2 + dxc * dxc + dyc * dyc);
    cur = c;
    grad = sgrad;
}

__device__ __forceinline__ void load_nbhd(const DevGeom& g, const float* img, int x0, int y0, float (&m)[4][4]) {
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int y = min(max(y0 - 1 + r, -PADR), g.ny + PADR - 1);
        const float* row = img + (size_t)(y + PADR) * g.pitch + PAD;       // one slice per image (DevGeom::sb == 1)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int x = min(x0 - 1 + c, g.nx + PAD - 1);
            m[r][c] = __ldg(row + x);
        }
    }
}

// the same neighbourhood in the two slices of a pair (images interleaved per pixel: one float2 per pixel)
__device__ __forceinline__ void load_nbhd2(const DevGeom& g, const float2* img2, int x0, int y0, float (&m0)[4][4], float (&m1)[4][4]) {
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int y = min(max(y0 - 1 + r, -PADR), g.ny + PADR - 1);
        const float2* row = img2 + (size_t)(y + PADR) * g.pitch + PAD;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int x = min(x0 - 1 + c, g.nx + PAD - 1);
            const float2 v = __ldg(row + x);
            m0[r][c] = v.x; m1[r][c] = v.y;
        }
    }
}

// atan(z) for |z| <= 0.75: odd polynomial, max error 3e-7 rad (fit on Chebyshev nodes; checked on the host side of
// the tests through the candidate-range parity cases)
__device__ __forceinline__ float atan_small(float z) {
    const float z2 = z * z;
    float p = -0.028348274528980255f;
    p = fmaf(p, z2, 0.08230143785476685f);
    p = fmaf(p, z2, -0.13596512377262115f);
    p = fmaf(p, z2, 0.19924239814281464f);
    p = fmaf(p, z2, -0.33330586552619934f);
    p = p * z2;
    return fmaf(z, p, z);
}

// K2's accumulators: NS == 4: acc.p[h][px] = the pair (component 2h, component 2h+1) of pixel px = ty*2+tx;
// NS == 1: acc.s[px].
template <int NS> struct BackAcc;
template <> struct BackAcc<4> {
    uint64_t p[2][4];
    __device__ __forceinline__ void clear() {
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
            for (int x = 0; x < 4; ++x) p[h][x] = 0ull;
    }
    __device__ __forceinline__ float get(int m, int px) const {
        float lo, hi;
        unpack2(p[m >> 1][px], lo, hi);
        return (m & 1) ? hi : lo;
    }
};
template <> struct BackAcc<1> {
    float s[4];
    __device__ __forceinline__ void clear() { s[0] = s[1] = s[2] = s[3] = 0.f; }
    __device__ __forceinline__ float get(int, int px) const { return s[px]; }
};

// one candidate ray r = {alpha, beta, g0, hk} against the 2x2 tile whose first pixel has centred indices (xc0, yc0):
// the four chord weights (over h, which the residuals sv already carry) feed the tile's accumulators; with NS == 4
// the same weights serve the orbit's four residuals, and with SB == 2 the two slices of the block.
__device__ __forceinline__ void back_weights(const float4 r, float xc0, float yc0, float (&w)[4]) {
    const float q00 = fmaf(r.x, xc0, fmaf(r.y, yc0, r.z));
    const float q01 = q00 + r.x;          // (ty=0, tx=1)
    const float q10 = q00 + r.y;          // (ty=1, tx=0)
    const float q11 = q10 + r.x;
    w[0] = __saturatef(r.w - fabsf(q00));
    w[1] = __saturatef(r.w - fabsf(q01));
    w[2] = __saturatef(r.w - fabsf(q10));
    w[3] = __saturatef(r.w - fabsf(q11));
}
__device__ __forceinline__ void back_fma(const float (&w)[4], const float4 sv, BackAcc<4>& acc) {
    const uint64_t sxy = pack2(sv.x, sv.y), szw = pack2(sv.z, sv.w);
#pragma unroll
    for (int p = 0; p < 4; ++p) { ffma2(acc.p[0][p], sxy, w[p]); ffma2(acc.p[1][p], szw, w[p]); }
}
__device__ __forceinline__ void back_fma(const float (&w)[4], const float4 sv, BackAcc<1>& acc) {
#pragma unroll
    for (int p = 0; p < 4; ++p) acc.s[p] = fmaf(w[p], sv.x, acc.s[p]);
}
// the residuals of candidate u of one view for the SB slices of the block (NS == 1: the scalar in .x)
// (sp = the view's first candidate in each slice's residual rows, u = candidate)
template <int NS, int SB>
__device__ __forceinline__ void back_load(const float* const (&sp)[SB], int u, float4 (&sv)[SB]) {
#pragma unroll
    for (int j = 0; j < SB; ++j)
        sv[j] = NS == 4 ? __ldg(reinterpret_cast<const float4*>(sp[j]) + u) : make_float4(__ldg(sp[j] + u), 0.f, 0.f, 0.f);
}

// ------------------------------------------------------------------------------------------------
// K2: matched gather backprojection of the residuals written by K1 (+ step rule, TV gradient, Eq. 3 update,
// positivity clamp, best-image copy when MODE == 1).
// One block per SM-sized share of the base tiles (NS == 4: the 2x2-pixel tiles of the quadrant x,y < N/2): the tiles
// are numbered patch by patch (a patch = 8 x 4 tiles = 16 x 8 pixels, patches grouped 2 x 2) and dealt out in runs of
// `tpb` consecutive tiles, so that a block owns a compact piece of the image.  A block is tpb tiles x `shares` view
// shares: thread t works on tile t % tpb for the views of share t / tpb (NS == 4: share q takes quarter turn q & 3
// and every (shares/4)-th base view).  For every view the channels whose ray can cross the tile form the interval
// |c - c*| <= hw around the channel coordinate c* of the tile centre (every such ray passes within the tile's
// half-diagonal of the centre, so its fan angle differs from the centre's by at most asin(r/L) <= tile_hw/along
// channels); each candidate costs one 16-byte ray-table load and one residual load (NS == 4: the float4 of the
// view's orbit).  The shares' sums meet in shared memory in a fixed order; thread (tile, k) then finishes rotation
// k of the tile (TV gradient, update, stores).  The host sizes the grid to one block per SM (plan_back).
// ------------------------------------------------------------------------------------------------
// tile number -> patch (8 x 4 tiles; patches grouped 2 x 2, groups row-major) -> origin (x0, y0) of the 2x2-pixel tile
__device__ __forceinline__ void tile_origin(int T, int ngx, unsigned ngx_magic, int& x0, int& y0) {
    const int patch = T >> 5, w = T & 31;
    const int grp = patch >> 2, sub = patch & 3;
    const int gy = fastdiv(grp, ngx_magic), gx = grp - gy * ngx;
    // inside the patch a quarter-warp (8 lanes: the unit in which a 16-byte load is served) covers 4 x 2 tiles, the four
    // quarter-warps 2 x 2 such blocks: its lanes' candidate windows then lie closer together than along a row of 8 tiles
    const int wx = (w & 3) + ((w >> 3) & 1) * 4, wy = ((w >> 2) & 1) + (w >> 4) * 2;
    x0 = (((gx << 1) + (sub & 1)) * BK_WX + wx) * BK_TX;
    y0 = (((gy << 1) + (sub >> 1)) * BK_WY + wy) * BK_TY;
}

// Candidate interval of the tile at (x0, y0) in table view v: the channels whose ray can cross the tile form the interval
// |c - c*| <= hw around the channel coordinate c* of the tile centre (every such ray passes within tile_r of the centre,
// so its fan angle differs from the centre's by at most asin(r/L) <= tile_hw/along channels).  Packed as
// first channel | count << 20; an empty interval starts at C (the zero columns of the residuals).
__device__ __forceinline__ int tile_interval(const DevGeom& g, int x0, int y0, int v) {
    const float X = ((float)x0 - g.cx + 0.5f * (BK_TX - 1)) * g.pixel, Y = ((float)y0 - g.cy + 0.5f * (BK_TY - 1)) * g.pixel;
    const float2 cs = __ldg(&g.views[v]);
    // fan angle of the tile centre: tan(gamma*) = perp/along; along >= SAD - r_max > 0
    const float along = g.sad - fmaf(X, cs.x, Y * cs.y);
    const float perp = fmaf(X, cs.y, -Y * cs.x);
    const float rinv = __fdividef(1.f, along);
    const float z = perp * rinv;
    const float gam = g.use_atanf ? atanf(z) : atan_small(z);
    const float cstar = fmaf(gam, g.inv_dgamma, g.c_center);
    const float hw = fmaf(g.tile_hw, rinv, 0.05f);
    const int c_lo = min(max(0, (int)ceilf(cstar - hw)), g.C);
    const int c_hi = min(g.C - 1, (int)floorf(cstar + hw));
    return c_lo | (max(c_hi - c_lo + 1, 0) << 20);
}

// A0 for K2: the intervals of every (view, tile) once per handle and orbit size -- they depend on the geometry only, and
// worked out inside K2 they were a sixth of its instructions and most of its start-up path.  tab [V][ntiles].
// The bound of tile_interval is then narrowed to the tile's exact support: the first and last channel of it for which
// K2's own weight expression (back_weights, the same float operations on the same table entry) gives a non-zero weight
// to one of the tile's pixels; every candidate outside contributes exactly 0, so leaving it out changes no bit, and
// the candidate loop -- bound by the load path, two 16-byte loads per candidate -- gets about a fifth shorter.
__global__ void __launch_bounds__(256) k_build_intervals(DevGeom g, int ns, int ngx, unsigned ngx_magic, int ntiles, int* __restrict__ tab) {
    const int T = blockIdx.x * 256 + threadIdx.x, v = blockIdx.y;
    if (T >= ntiles) return;
    int x0, y0;
    tile_origin(T, ngx, ngx_magic, x0, y0);
    const int xlim = ns == 4 ? (g.nx >> 1) : g.nx, ylim = ns == 4 ? (g.ny >> 1) : g.ny;
    int packed = g.C;
    if (x0 < xlim && y0 < ylim) {
        const int loose = tile_interval(g, x0, y0, v);
        const int c_lo = loose & 0xfffff, n = loose >> 20;
        const float xc0 = (float)x0 - g.cx, yc0 = (float)y0 - g.cy;
        int first = -1, last = -1;
        for (int u = 0; u < n; ++u) {
            float w[4];
            back_weights(__ldg(&g.rays[(size_t)v * g.C + c_lo + u]), xc0, yc0, w);
            if (w[0] > 0.f || w[1] > 0.f || w[2] > 0.f || w[3] > 0.f) { if (first < 0) first = u; last = u; }
        }
        if (first >= 0) packed = (c_lo + first) | ((last - first + 1) << 20);
    }
    tab[(size_t)v * ntiles + T] = packed;
}

// STACK == 1 (SB == 1 only): the slices of the launch form a volume (readings H1-H3) -- per-slice view shift and the z
// term of the 3-D TV; kept out of the default instantiation, whose registers are tight.
template <int MODE, int NS, int SB, int STACK>
__global__ void __launch_bounds__(SB == 1 ? BK_MAX_THREADS : BKB_MAX_THREADS, SB == 1 ? 1 : 2) k_back(const BackArgs a) {
    const DevGeom& g = a.g;
    const int t = threadIdx.x, lane = t & 31, s0 = blockIdx.z * SB;       // slices s0 .. s0 + SB - 1
    OSIV_TL(a.iter, 1, 0, false);
    const int tpb = a.tpb, shares = a.shares;
    const int q = fastdiv(t, a.tpb_magic), i = t - q * tpb;
    extern __shared__ float red[];                        // NS == 4: [SB][4 pixels][shares][tpb] float4 (the 4 rotations); NS == 1: [SB][shares][4][tpb]

    const int xlim = NS == 4 ? (g.nx >> 1) : g.nx, ylim = NS == 4 ? (g.ny >> 1) : g.ny;
    int x0, y0;
    const int T = blockIdx.x * tpb + i;
    tile_origin(T, a.ngx, a.ngx_magic, x0, y0);
    const bool active = q < shares && x0 < xlim && y0 < ylim;

    // acc[m][ty*2+tx]: NS == 4: m = component of the orbit's residual float4 (this thread's views all lie in quarter
    // turn `quarter`, so rotation k of the tile collects component (quarter + k) % 4)
    BackAcc<NS> acc[SB];
#pragma unroll
    for (int j = 0; j < SB; ++j) acc[j].clear();

    OSIV_TL(a.iter, 1, 7, false);
    const int VSb = a.VS / NS;
    const int vshift = STACK ? (int)(((unsigned)a.view_shift * (unsigned)s0) % (unsigned)g.V) : 0;
    const int quarter = NS == 4 ? (q & 3) : 0;
    const int jfirst = NS == 4 ? (q >> 2) : q, jstep = NS == 4 ? (shares >> 2) : shares;
    const int ntrips = (VSb + jstep - 1) / jstep;         // the same for every thread: the candidate loop is warp-wide
    {
        const float xc0 = (float)x0 - g.cx, yc0 = (float)y0 - g.cy;
        const float* res[SB];                                    // same float count for both layouts; a slice past the
#pragma unroll
        for (int j = 0; j < SB; ++j) res[j] = a.res + (size_t)(SB == 1 ? s0 : min(s0 + j, a.batch - 1)) * a.VS * a.Cp;   // batch repeats the last

        // Candidate interval of trip `it` (view jfirst + it * jstep of this thread's share): offsets of its first
        // candidate in the ray table and in the residual rows, and the warp's candidate count.  The warp runs
        // max-over-lanes candidates in lock step (no remainder code); a lane's extra candidates have zero weight (the
        // ray misses its tile) or read the zero columns C..Cp-1 of res, and a lane that is off reads only those.
        // Trips are taken four at a time.  Their packed intervals are plain loads from the table (unconditional, index
        // clamped: four loads in flight, nothing from K1 needed, so the first four are fetched and decoded before the
        // wait, and the next four while the current ones are walked); the candidates of two trips are then walked
        // together, which keeps 2 x 2 x 2 sixteen-byte loads in flight per thread.
        const int Tc = min(T, a.ntiles - 1);
        auto trip_view = [&](int it, int& jb) -> int {           // table view of trip `it` of this thread's share
            jb = min(jfirst + it * jstep, VSb - 1);
            const int jj = jb + quarter * VSb;
            int v = a.subset < 0 ? jj : a.subset + jj * a.M;
            if (STACK) { v += vshift; if (v >= g.V) v -= g.V; }      // H1
            return v;
        };
        auto fetch = [&](int it) -> int {                        // k_build_intervals' entry, or "empty" (first channel C, count 0)
            int jb;
            const int v = trip_view(it, jb);
            const int pk = __ldg(&a.itab[(size_t)v * a.ntiles + Tc]);
            return (active && jfirst + it * jstep < VSb) ? pk : g.C;
        };
        auto decode = [&](int it, int pk, int& offR, int& offS) -> int {
            int jb;
            const int v = trip_view(it, jb);
            const int c_lo = pk & 0xfffff;
            offR = v * g.C + c_lo;
            offS = jb * a.Cp + c_lo;
            return __reduce_max_sync(0xffffffffu, pk >> 20);
        };
        constexpr int CH = 4;
        int offR[CH], offS[CH], ncw[CH], pk[CH];
#pragma unroll
        for (int e = 0; e < CH; ++e) pk[e] = e < ntrips ? fetch(e) : g.C;
#pragma unroll
        for (int e = 0; e < CH; ++e) {
            ncw[e] = decode(e, pk[e], offR[e], offS[e]);
            pdl_before_wait(ncw[e]);
        }
        OSIV_TL(a.iter, 1, 1, false);
        pdl_wait();                                              // the residuals are the previous launch's output
        pdl_launch_next();
        OSIV_TL(a.iter, 1, 2, false);
        for (int it0 = 0;;) {
            const bool more = it0 + CH < ntrips;                 // warp-uniform
            if (more) {
#pragma unroll
                for (int e = 0; e < CH; ++e) pk[e] = it0 + CH + e < ntrips ? fetch(it0 + CH + e) : g.C;
            }
#pragma unroll
            for (int e = 0; e < CH; e += 2) {
                const float4* rpA = g.rays + offR[e];
                const float4* rpB = g.rays + offR[e + 1];
                if constexpr (SB == 1) {                   // one slice: plain pointers (the register budget is tight)
                    const float4* spA = reinterpret_cast<const float4*>(res[0]) + offS[e];      // NS == 4
                    const float4* spB = reinterpret_cast<const float4*>(res[0]) + offS[e + 1];
                    const float* tpA = res[0] + offS[e];                                        // NS == 1
                    const float* tpB = res[0] + offS[e + 1];
                    if (ncw[e + 1] == 0) {                 // odd trip out (warp-uniform): one stream
#pragma unroll 2
                        for (int u = 0; u < ncw[e]; ++u) {
                            const float4 rA = __ldg(rpA + u);
                            const float4 sA = NS == 4 ? __ldg(spA + u) : make_float4(__ldg(tpA + u), 0.f, 0.f, 0.f);
                            float wA[4];
                            back_weights(rA, xc0, yc0, wA);
                            back_fma(wA, sA, acc[0]);
                        }
                    } else {
                        const int n = max(ncw[e], ncw[e + 1]);
#pragma unroll 2
                        for (int u = 0; u < n; ++u) {
                            OSIV_CHECK(offR[e] + u < a.ray_entries && offR[e + 1] + u < a.ray_entries, 4);
                            OSIV_CHECK((long long)(offS[e] + u + 1) * NS <= (long long)a.VS * a.Cp && (long long)(offS[e + 1] + u + 1) * NS <= (long long)a.VS * a.Cp, 5);
                            const float4 rA = __ldg(rpA + u), rB = __ldg(rpB + u);
                            const float4 sA = NS == 4 ? __ldg(spA + u) : make_float4(__ldg(tpA + u), 0.f, 0.f, 0.f);
                            const float4 sB = NS == 4 ? __ldg(spB + u) : make_float4(__ldg(tpB + u), 0.f, 0.f, 0.f);
                            float wA[4], wB[4];
                            back_weights(rA, xc0, yc0, wA);
                            back_fma(wA, sA, acc[0]);
                            back_weights(rB, xc0, yc0, wB);
                            back_fma(wB, sB, acc[0]);
                        }
                    }
                } else {
                    const float* spA[SB];
                    const float* spB[SB];
#pragma unroll
                    for (int j = 0; j < SB; ++j) {
                        spA[j] = res[j] + (size_t)offS[e] * NS;          // NS == 4: float4 entries
                        spB[j] = res[j] + (size_t)offS[e + 1] * NS;
                    }
                    if (ncw[e + 1] == 0) {                 // odd trip out (warp-uniform): one stream
#pragma unroll 2
                        for (int u = 0; u < ncw[e]; ++u) {
                            const float4 rA = __ldg(rpA + u);
                            float4 sA[SB];
                            back_load<NS, SB>(spA, u, sA);
                            float wA[4];
                            back_weights(rA, xc0, yc0, wA);
#pragma unroll
                            for (int j = 0; j < SB; ++j) back_fma(wA, sA[j], acc[j]);
                        }
                    } else {
                        const int n = max(ncw[e], ncw[e + 1]);
#pragma unroll 2
                        for (int u = 0; u < n; ++u) {
                            const float4 rA = __ldg(rpA + u), rB = __ldg(rpB + u);
                            float4 sA[SB], sB[SB];
                            back_load<NS, SB>(spA, u, sA);
                            back_load<NS, SB>(spB, u, sB);
                            float wA[4], wB[4];
                            back_weights(rA, xc0, yc0, wA);
                            back_weights(rB, xc0, yc0, wB);
#pragma unroll
                            for (int j = 0; j < SB; ++j) { back_fma(wA, sA[j], acc[j]); back_fma(wB, sB[j], acc[j]); }
                        }
                    }
                }
            }
            if (!more) break;
            it0 += CH;
#pragma unroll
            for (int e = 0; e < CH; ++e) ncw[e] = decode(it0 + e, pk[e], offR[e], offS[e]);
        }
    }
    OSIV_TL(a.iter, 1, 3, true);
    // The shares' sums meet in shared memory: red[slice j][share q][rotation k][pixel p][tile i]; rotation k of the tile
    // collects component (quarter + k) % 4 of the orbit's residuals  <=>  component m feeds rotation (m - quarter) % 4.
    if (q < shares) {
#pragma unroll
        for (int j = 0; j < SB; ++j) {
            if constexpr (NS == 4) {
                float4* red4 = reinterpret_cast<float4*>(red);
#pragma unroll
                for (int p = 0; p < 4; ++p) {
                    float r4[4];
#pragma unroll
                    for (int m = 0; m < 4; ++m) r4[(m - quarter) & 3] = acc[j].get(m, p);
                    red4[((j * 4 + p) * shares + q) * tpb + i] = make_float4(r4[0], r4[1], r4[2], r4[3]);
                }
            } else {
#pragma unroll
                for (int p = 0; p < 4; ++p) red[((j * shares + q) * 4 + p) * tpb + i] = acc[j].get(0, p);
            }
        }
    }
    const bool tile_ok = x0 < xlim && y0 < ylim;

    if constexpr (NS == 4) {
        // ---- quarter-turn path: thread (tile i, p = q < 4) finishes base pixel p of the tile in all four rotations.
        // Everything that does not depend on the other shares' sums -- monitor, step rule, the 3x3 neighbourhood of
        // float4s of mu(n) (= the neighbourhoods of all four rotated pixels), TV gradient -- is done before the
        // barrier, so that its loads overlap the wait for the slowest warp.
        const bool fin_active = q < 4 && tile_ok;
        const int N = g.nx;
        const int px = x0 + (q & 1), py = y0 + ((q >> 1) & 1);      // base pixel P (q < 4)
        StepInfo si[SB];
        float step[SB], cur[SB][4], tv[SB][4];
        if (MODE == 1 && t < 32 * ((4 * tpb + 31) / 32)) {           // whole warps: step_rule shuffles
            const bool writer = blockIdx.x == 0 && t < 32;
#pragma unroll
            for (int j = 0; j < SB; ++j) {
                const int s = s0 + j;
                if (s >= a.batch) break;
                float4 E[3][3];
                if (fin_active) {
                    const float4* Q = reinterpret_cast<const float4*>(a.img) + (size_t)(blockIdx.z * SB + j) * g.img_elems;
#pragma unroll
                    for (int dy = 0; dy < 3; ++dy)
#pragma unroll
                        for (int dx = 0; dx < 3; ++dx) E[dy][dx] = __ldg(Q + (size_t)((py + dy - 1 + PADR) * g.pitch + PAD + px + dx - 1));
                }
                si[j] = step_rule(a, s, lane, writer);
                step[j] = (float)(si[j].lambda * a.tau);
                if (fin_active) {                                    // A5 for R^k P, k = 0..3
                    if (px > 0 && py > 0) {                          // off the image border (P lies in the base quadrant)
                        orbit_tv_inner<0>(E, a.eps2, cur[j][0], tv[j][0]);
                        orbit_tv_inner<1>(E, a.eps2, cur[j][1], tv[j][1]);
                        orbit_tv_inner<2>(E, a.eps2, cur[j][2], tv[j][2]);
                        orbit_tv_inner<3>(E, a.eps2, cur[j][3], tv[j][3]);
                    } else {
                        orbit_tv<0>(E, px, py, N, a.eps2, cur[j][0], tv[j][0]);
                        orbit_tv<1>(E, px, py, N, a.eps2, cur[j][1], tv[j][1]);
                        orbit_tv<2>(E, px, py, N, a.eps2, cur[j][2], tv[j][2]);
                        orbit_tv<3>(E, px, py, N, a.eps2, cur[j][3], tv[j][3]);
                    }
                }
            }
        }
        __syncthreads();
        OSIV_TL(a.iter, 1, 4, false);
        if (!fin_active) return;
        // the four rotated positions of P: R^k P
        const int rx[4] = {px, N - 1 - py, N - 1 - px, py}, ry[4] = {py, px, N - 1 - py, N - 1 - px};
#pragma unroll
        for (int j = 0; j < SB; ++j) {
            const int s = s0 + j;
            if (s >= a.batch) break;
            float gsum[4] = {0.f, 0.f, 0.f, 0.f};                    // g at R^k P: sums over the view shares, fixed order
            const float4* rp = reinterpret_cast<const float4*>(red) + (size_t)(j * 4 + q) * shares * tpb + i;
#pragma unroll 4
            for (int qq = 0; qq < shares; ++qq, rp += tpb) {
                const float4 v = *rp;
                gsum[0] += v.x; gsum[1] += v.y; gsum[2] += v.z; gsum[3] += v.w;
            }
            if constexpr (MODE == 0) {
                float* out = a.out + (size_t)s * N * N;
#pragma unroll
                for (int k = 0; k < 4; ++k) out[(size_t)ry[k] * N + rx[k]] = gsum[k];
            } else {
            // ---- A6 update (Eq. 3) with mu > 0; the new float4 of R^k P is the orbit read from k on
            float un[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) un[k] = fmaxf(fmaf(step[j], gsum[k] - a.beta_over_M * tv[j][k], cur[j][k]), 0.f);
            float4* Qn = reinterpret_cast<float4*>(a.img_new) + (size_t)(blockIdx.z * SB + j) * g.img_elems;
            float4* QTn = reinterpret_cast<float4*>(a.imgT_new) + (size_t)(blockIdx.z * SB + j) * g.imgT_elems;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const float4 v = make_float4(un[k], un[(k + 1) & 3], un[(k + 2) & 3], un[(k + 3) & 3]);
                Qn[pad_off(g, ry[k], rx[k])] = v;
                QTn[padT_off(g, rx[k], ry[k])] = v;
            }
            if (a.best && si[j].improved) {                          // A7: mu(n) had the smallest monitor so far
                float* best = a.best + (size_t)s * N * N;
#pragma unroll
                for (int k = 0; k < 4; ++k) best[(size_t)ry[k] * N + rx[k]] = cur[j][k];
            }
            }
        }
        OSIV_TL(a.iter, 1, 5, true);
    } else if constexpr (SB == 1) {                        // general path, one slice per block: scalars (the register budget is tight)
        const int s = s0;
        // thread (tile i, share 0) finishes the tile.  Everything that does not depend on the other shares' sums --
        // monitor, step rule, neighbourhood of mu(n), TV gradient -- is done before the barrier, so that its loads
        // overlap the wait for the slowest warp.
        const bool fin_active = q == 0 && tile_ok;
        StepInfo si;
        float step = 0.f;
        float m[4][4], tv[2][2];
        if (MODE == 1 && t < 32 * ((tpb + 31) / 32)) {               // whole warps: step_rule shuffles
            const bool writer = blockIdx.x == 0 && t < 32;
            if (fin_active) load_nbhd(g, a.img + (size_t)s * g.img_elems, x0, y0, m);
            si = step_rule(a, s, lane, writer);
            step = (float)(si.lambda * a.tau);
            if (fin_active) {
                if (STACK && a.tv_z > 0.f) {                        // stack of slices: the z term needs slices s-1 and s+1
                    const bool has_up = s + 1 < a.batch, has_dn = s > 0;
                    float up[4][4], dn[4][4];
                    load_nbhd(g, a.img + (size_t)(has_up ? s + 1 : s) * g.img_elems, x0, y0, up);
                    load_nbhd(g, a.img + (size_t)(has_dn ? s - 1 : s) * g.img_elems, x0, y0, dn);
                    tv_grad_tile3(m, up, dn, has_up, has_dn, a.tv_z, x0, y0, g.nx, g.ny, a.eps2, tv);
                } else {
                    tv_grad_tile(m, x0, y0, g.nx, g.ny, a.eps2, tv);
                }
            }
        }
        __syncthreads();
        if (!fin_active) return;
        float b[4];                                                  // sums over the view shares, fixed order
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            float x = 0.f;
            for (int qq = 0; qq < shares; ++qq) x += red[(qq * 4 + p) * tpb + i];
            b[p] = x;
        }
        const bool vx1 = x0 + 1 < g.nx, vy1 = y0 + 1 < g.ny;
        if (MODE == 0) {
            float* out = a.out + (size_t)s * g.nx * g.ny;
            out[(size_t)y0 * g.nx + x0] = b[0];
            if (vx1) out[(size_t)y0 * g.nx + x0 + 1] = b[1];
            if (vy1) out[(size_t)(y0 + 1) * g.nx + x0] = b[2];
            if (vx1 && vy1) out[(size_t)(y0 + 1) * g.nx + x0 + 1] = b[3];
            return;
        }
        // ---- A5 TV gradient of mu(n), A6 update (Eq. 3) with mu > 0, A7 best copy ----
        const float u00 = fmaxf(fmaf(step, b[0] - a.beta_over_M * tv[0][0], m[1][1]), 0.f);
        const float u01 = fmaxf(fmaf(step, b[1] - a.beta_over_M * tv[0][1], m[1][2]), 0.f);
        const float u10 = fmaxf(fmaf(step, b[2] - a.beta_over_M * tv[1][0], m[2][1]), 0.f);
        const float u11 = fmaxf(fmaf(step, b[3] - a.beta_over_M * tv[1][1], m[2][2]), 0.f);
        float* nimg = a.img_new + (size_t)s * g.img_elems;
        float* nimgT = a.imgT_new + (size_t)s * g.imgT_elems;
        nimg[pad_off(g, y0, x0)] = u00;
        nimgT[padT_off(g, x0, y0)] = u00;
        if (vx1) { nimg[pad_off(g, y0, x0 + 1)] = u01; nimgT[padT_off(g, x0 + 1, y0)] = u01; }
        if (vy1) { nimg[pad_off(g, y0 + 1, x0)] = u10; nimgT[padT_off(g, x0, y0 + 1)] = u10; }
        if (vx1 && vy1) { nimg[pad_off(g, y0 + 1, x0 + 1)] = u11; nimgT[padT_off(g, x0 + 1, y0 + 1)] = u11; }
        if (a.best && si.improved) {
            float* best = a.best + (size_t)s * g.nx * g.ny;
            best[(size_t)y0 * g.nx + x0] = m[1][1];
            if (vx1) best[(size_t)y0 * g.nx + x0 + 1] = m[1][2];
            if (vy1) best[(size_t)(y0 + 1) * g.nx + x0] = m[2][1];
            if (vx1 && vy1) best[(size_t)(y0 + 1) * g.nx + x0 + 1] = m[2][2];
        }
    } else {                                               // general path, a pair of slices per block (images interleaved per pixel)
        const bool fin_active = q == 0 && tile_ok;
        StepInfo si[SB];
        float step[SB], m[SB][4][4], tv[SB][2][2];
        if (MODE == 1 && t < 32 * ((tpb + 31) / 32)) {               // whole warps: step_rule shuffles
            const bool writer = blockIdx.x == 0 && t < 32;
            if (fin_active) load_nbhd2(g, reinterpret_cast<const float2*>(a.img) + (size_t)blockIdx.z * g.img_elems, x0, y0, m[0], m[SB - 1]);
#pragma unroll
            for (int j = 0; j < SB; ++j) {
                const int s = s0 + j;
                if (s >= a.batch) break;
                si[j] = step_rule(a, s, lane, writer);
                step[j] = (float)(si[j].lambda * a.tau);
                if (fin_active) tv_grad_tile(m[j], x0, y0, g.nx, g.ny, a.eps2, tv[j]);
            }
        }
        __syncthreads();
        if (!fin_active) return;
        float un[SB][4] = {};                                     // mu(n+1) of the tile in both slices (0 in an empty one)
        const bool vx1 = x0 + 1 < g.nx, vy1 = y0 + 1 < g.ny;
#pragma unroll
        for (int j = 0; j < SB; ++j) {
            const int s = s0 + j;
            if (s >= a.batch) break;
            float b[4];                                           // sums over the view shares, fixed order
#pragma unroll
            for (int p = 0; p < 4; ++p) {
                float x = 0.f;
                for (int qq = 0; qq < shares; ++qq) x += red[((j * shares + qq) * 4 + p) * tpb + i];
                b[p] = x;
            }
            if (MODE == 0) {
                float* out = a.out + (size_t)s * g.nx * g.ny;
                out[(size_t)y0 * g.nx + x0] = b[0];
                if (vx1) out[(size_t)y0 * g.nx + x0 + 1] = b[1];
                if (vy1) out[(size_t)(y0 + 1) * g.nx + x0] = b[2];
                if (vx1 && vy1) out[(size_t)(y0 + 1) * g.nx + x0 + 1] = b[3];
                continue;
            }
            un[j][0] = fmaxf(fmaf(step[j], b[0] - a.beta_over_M * tv[j][0][0], m[j][1][1]), 0.f);
            un[j][1] = fmaxf(fmaf(step[j], b[1] - a.beta_over_M * tv[j][0][1], m[j][1][2]), 0.f);
            un[j][2] = fmaxf(fmaf(step[j], b[2] - a.beta_over_M * tv[j][1][0], m[j][2][1]), 0.f);
            un[j][3] = fmaxf(fmaf(step[j], b[3] - a.beta_over_M * tv[j][1][1], m[j][2][2]), 0.f);
            if (a.best && si[j].improved) {
                float* best = a.best + (size_t)s * g.nx * g.ny;
                best[(size_t)y0 * g.nx + x0] = m[j][1][1];
                if (vx1) best[(size_t)y0 * g.nx + x0 + 1] = m[j][1][2];
                if (vy1) best[(size_t)(y0 + 1) * g.nx + x0] = m[j][2][1];
                if (vx1 && vy1) best[(size_t)(y0 + 1) * g.nx + x0 + 1] = m[j][2][2];
            }
        }
        if constexpr (MODE == 1) {
            float2* nimg = reinterpret_cast<float2*>(a.img_new) + (size_t)blockIdx.z * g.img_elems;
            float2* nimgT = reinterpret_cast<float2*>(a.imgT_new) + (size_t)blockIdx.z * g.imgT_elems;
            const float2 u00 = make_float2(un[0][0], un[SB - 1][0]), u01 = make_float2(un[0][1], un[SB - 1][1]);
            const float2 u10 = make_float2(un[0][2], un[SB - 1][2]), u11 = make_float2(un[0][3], un[SB - 1][3]);
            nimg[pad_off(g, y0, x0)] = u00;
            nimgT[padT_off(g, x0, y0)] = u00;
            if (vx1) { nimg[pad_off(g, y0, x0 + 1)] = u01; nimgT[padT_off(g, x0 + 1, y0)] = u01; }
            if (vy1) { nimg[pad_off(g, y0 + 1, x0)] = u10; nimgT[padT_off(g, x0, y0 + 1)] = u10; }
            if (vx1 && vy1) { nimg[pad_off(g, y0 + 1, x0 + 1)] = u11; nimgT[padT_off(g, x0 + 1, y0 + 1)] = u11; }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Small helpers around the two hot kernels
// ------------------------------------------------------------------------------------------------

// Image layouts of the padded working buffers (NS == 1: per group of g.sb slices, slices interleaved per pixel; NS == 4: slice-major):
//   NS == 1: one float per pixel and slice:   img[((iy+PADR)*pitch + PAD+ix) * sb + sl],  imgT the transpose;
//   NS == 4: one float4 per pixel and slice:  Q  [sl][(iy+PADR)*pitch + PAD+ix] = {mu(P), mu(RP), mu(R^2P), mu(R^3P)},
//            R: (ix,iy) -> (N-1-iy, ix);  QT the transpose.
__device__ __forceinline__ void orbit_pos(int N, int ix, int iy, int k, int& x, int& y) {
    x = k == 0 ? ix : k == 1 ? N - 1 - iy : k == 2 ? N - 1 - ix : iy;
    y = k == 0 ? iy : k == 1 ? ix : k == 2 ? N - 1 - iy : N - 1 - ix;
}

// [batch][ny][nx] -> the padded working layout and its transpose
__global__ void __launch_bounds__(256) k_pad_transpose(DevGeom g, int ns, const float* __restrict__ src,
                                                       float* __restrict__ img, float* __restrict__ imgT) {
    const int s = blockIdx.z;
    const int x = blockIdx.x * 32 + (threadIdx.x & 31);
    const int y = blockIdx.y * 8 + (threadIdx.x >> 5);
    if (x >= g.nx || y >= g.ny) return;
    src += (size_t)s * g.nx * g.ny;
    if (ns == 4) {
        float v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) { int xx, yy; orbit_pos(g.nx, x, y, k, xx, yy); v[k] = src[(size_t)yy * g.nx + xx]; }
        const float4 q = make_float4(v[0], v[1], v[2], v[3]);
        reinterpret_cast<float4*>(img)[(size_t)s * g.img_elems + pad_off(g, y, x)] = q;
        reinterpret_cast<float4*>(imgT)[(size_t)s * g.imgT_elems + padT_off(g, x, y)] = q;
    } else {
        const float v = src[(size_t)y * g.nx + x];
        img[slice_base(g, g.img_elems, s) + pad_off(g, y, x) * g.sb] = v;
        imgT[slice_base(g, g.imgT_elems, s) + padT_off(g, x, y) * g.sb] = v;
    }
}

// working layout -> [batch][ny][nx]; with best != null picks per slice: improved ? img : best   (C12)
__global__ void __launch_bounds__(256) k_unpad(DevGeom g, int ns, const float* __restrict__ img,
                                               const float* __restrict__ best, const SliceState* __restrict__ state,
                                               float* __restrict__ out) {
    const int s = blockIdx.z;
    const int x = blockIdx.x * 32 + (threadIdx.x & 31);
    const int y = blockIdx.y * 8 + (threadIdx.x >> 5);
    if (x >= g.nx || y >= g.ny) return;
    const size_t o = (size_t)s * g.nx * g.ny + (size_t)y * g.nx + x;
    if (best && !state[s].improved) out[o] = best[o];
    else if (ns == 4) out[o] = reinterpret_cast<const float4*>(img)[(size_t)s * g.img_elems + pad_off(g, y, x)].x;
    else out[o] = img[slice_base(g, g.img_elems, s) + pad_off(g, y, x) * g.sb];
}

// homogeneous initial image into both working layouts, and into best
__global__ void __launch_bounds__(256) k_fill(DevGeom g, int ns, float mu0, float* __restrict__ img,
                                              float* __restrict__ imgT, float* __restrict__ best) {
    const int s = blockIdx.z;
    const int x = blockIdx.x * 32 + (threadIdx.x & 31);
    const int y = blockIdx.y * 8 + (threadIdx.x >> 5);
    if (x >= g.nx || y >= g.ny) return;
    if (ns == 4) {
        const float4 q = make_float4(mu0, mu0, mu0, mu0);
        reinterpret_cast<float4*>(img)[(size_t)s * g.img_elems + pad_off(g, y, x)] = q;
        reinterpret_cast<float4*>(imgT)[(size_t)s * g.imgT_elems + padT_off(g, x, y)] = q;
    } else {
        img[slice_base(g, g.img_elems, s) + pad_off(g, y, x) * g.sb] = mu0;
        imgT[slice_base(g, g.imgT_elems, s) + padT_off(g, x, y) * g.sb] = mu0;
    }
    if (best) best[(size_t)s * g.nx * g.ny + (size_t)y * g.nx + x] = mu0;
}

// per-slice state reset and 1/b_ref, b_ref = mean_c b_c (one warp, fixed order)
__global__ void k_init_state(SliceState* state, int* not_finite, int batch, double lambda0, const float* blank,
                             float blank_scalar, int C, float* inv_bref) {
    const int lane = threadIdx.x;
    for (int s = lane; s < batch; s += 32) {
        SliceState st;
        st.lambda = lambda0; st.D_prev = 0.0; st.D_best = __longlong_as_double(0x7ff0000000000000LL);
        st.D_last = 0.0; st.n = 0; st.improved = 0; st.pad0 = 0; st.pad1 = 0;
        state[s] = st;
        not_finite[s] = 0;
    }
    double sum = 0.0;
    if (blank) {
        for (int c = lane; c < C; c += 32) sum += (double)blank[c];
        for (int off = 16; off > 0; off >>= 1) sum += __shfl_down_sync(0xffffffffu, sum, off);
        sum /= (double)C;
    } else {
        sum = (double)blank_scalar;
    }
    if (lane == 0) *inv_bref = (float)(1.0 / sum);
}

// sinogram [batch][VS][C] -> h * s in the layout of FwdArgs::res, for the standalone backprojection
__global__ void __launch_bounds__(256) k_scale_sino(DevGeom g, const float* __restrict__ sino, float* __restrict__ res,
                                                    int subset, int M, int VS, int ns, int Cp) {
    const int c = blockIdx.x * 256 + threadIdx.x, j = blockIdx.y, s = blockIdx.z;
    if (c >= g.C) return;
    const int v = subset < 0 ? j : subset + j * M;
    const float val = __ldg(&g.hs[(size_t)v * g.C + c]) * sino[((size_t)s * VS + j) * g.C + c];
    if (ns == 4) {
        const int VSb = VS / 4, jb = j % VSb, k = j / VSb;
        res[(((size_t)s * VSb + jb) * Cp + c) * 4 + k] = val;
    } else {
        res[((size_t)s * VS + j) * Cp + c] = val;
    }
}

// standalone TV gradient: [batch][ny][nx] -> [batch][ny][nx] through the padded workspace
__global__ void __launch_bounds__(128) k_tv(DevGeom g, const float* __restrict__ img, float eps2,
                                            float* __restrict__ out) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int x0 = (blockIdx.x * 16 + (warp & 1) * 8 + (lane & 7)) * 2;
    const int y0 = (blockIdx.y * 8 + (warp >> 1) * 4 + (lane >> 3)) * 2;
    const int s = blockIdx.z;
    if (x0 >= g.nx || y0 >= g.ny) return;
    float m[4][4], tv[2][2];
    load_nbhd(g, img + (size_t)s * g.img_elems, x0, y0, m);
    tv_grad_tile(m, x0, y0, g.nx, g.ny, eps2, tv);
    out += (size_t)s * g.nx * g.ny;
    const bool vx1 = x0 + 1 < g.nx, vy1 = y0 + 1 < g.ny;
    out[(size_t)y0 * g.nx + x0] = tv[0][0];
    if (vx1) out[(size_t)y0 * g.nx + x0 + 1] = tv[0][1];
    if (vy1) out[(size_t)(y0 + 1) * g.nx + x0] = tv[1][0];
    if (vx1 && vy1) out[(size_t)(y0 + 1) * g.nx + x0 + 1] = tv[1][1];
}

}  // namespace osiv
