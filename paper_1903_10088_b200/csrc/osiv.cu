// osiv.cu -- host side of libosiv: the C ABI of include/osiv.h over the kernels in osiv_kernels.cuh.
// Build: nvcc -O3 -lineinfo -gencode arch=compute_100a,code=sm_100a -shared -Xcompiler -fPIC
// (paper_1903_10088_b200/build.py).  No CPU fallback exists: without a usable device every
// compute entry point returns OSIV_ERR_CUDA.
#include "../../include/osiv.h"
#include "osiv_kernels.cuh"
#include "osiv_back_staged.cuh"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

using namespace osiv;

struct osiv_handle {
    osiv_geometry geom;
    double dgamma;
    int device;
    int max_batch;
    DevGeom dg;
    float4* d_rays = nullptr;
    float2* d_views = nullptr;
    float* d_hs = nullptr;
    // per-slice workspace, grown lazily
    int ws_batch = 0, ws_sb = 1, ws_ns = 1;   // slices the image buffers hold, their interleave (DevGeom::sb) and layout (1: one
                                              // float per pixel, 4: the orbit float4 per pixel of the quarter-turn path)
    float *d_imgA = nullptr, *d_imgB = nullptr, *d_imgTA = nullptr, *d_imgTB = nullptr;
    float* d_best = nullptr;
    size_t res_elems = 0;       float* d_res = nullptr;
    long long res_key = -1;             // layout (V_S, orbit size, batch) whose zero columns d_res currently holds
    int res_pad = 4;                    // zero columns C..Cp-1 of every residual row (K2 reads past a tile's last candidate)
    size_t dpart_elems = 0;     double* d_dparts = nullptr;
    int* d_itab[2] = {nullptr, nullptr};    // K2's candidate intervals [V][ntiles], built on first use; [0]: NS = 1, [1]: NS = 4
    int itab_tiles[2] = {0, 0};
    SliceState* d_state = nullptr;      // [2][max_batch], ping-pong between iterations
    int* d_not_finite = nullptr;        // [max_batch]
    float* d_inv_bref = nullptr;
    int num_sms = 148;
    size_t trace_elems = 0;     double* d_trace = nullptr;
    size_t forced_elems = 0;    double* d_forced = nullptr;
    size_t dhist_elems = 0;     double* d_dhist = nullptr;
    // staging for osiv_reconstruct_host
    size_t hc_elems = 0;        float* d_hcounts = nullptr;
    float* d_hblank = nullptr;
    size_t hi_elems = 0;        float* d_himg = nullptr;
    int64_t launches = 0;
    int force_ns1 = 0;                  // osiv_set_symmetry(h, 0): always take the general path
    long long ray_entries = 0;          // float4 entries behind d_rays (table + zero slack)
    // staged K2 (osiv_back_staged.cuh): regions of the base quadrant, per-(view, block) windows, per-tile intervals
    int st_ready = 0;                   // 1: tables built and usable; 0: this geometry does not take the staged kernel
    int st_off = 0;                     // osiv_set_back_kernel: 0 = staged when one round suffices, 1 = always the general K2, 2 = staged
    std::vector<int4> st_regions;       // host copy of d_regions (passed in the kernel parameters when short enough)
                                        // whenever the geometry allows (several rounds)
    int st_nblk = 0, st_tpbp = 0, st_W = 0;
    int4* d_regions = nullptr;
    unsigned short* d_itab2 = nullptr;
    int* d_bwin = nullptr;
    float* d_invk = nullptr;            // [V][C] 1 / (in-line coefficient) of every ray (K1's start-up path)
    int4* d_k1rng = nullptr;            // K1's block line ranges for (k1rng_M subsets, orbit size, rays per block), k_build_fwd_ranges
    size_t k1rng_elems = 0;
    long long k1rng_key = -1;
    std::vector<unsigned short> k1order; // [M][blocks]: K1's runs of rays, longest walk first (FwdArgs::order), with d_k1rng
    unsigned char* d_blob = nullptr;    // per-subset constants of the staged K2 for blob_M subsets (k_build_blob)
    size_t blob_bytes = 0;
    int blob_M = 0;
    int use_pdl = 1;                    // osiv_set_overlap(h, 0): plain stream order between K1 and K2
    // the launch sequence of one osiv_reconstruct call as a CUDA graph, replayed while the call's arguments repeat
    int use_graph = 1;                  // osiv_set_graph(h, 0): enqueue every launch from the host
    cudaStream_t cap_stream = nullptr;  // capture happens here (the caller's stream may be the legacy default stream)
    struct GraphSlot {                  // two argument sets are remembered (a caller alternating between the device-pointer and
        std::vector<unsigned char> key; //  the host-buffer entry point keeps both graphs)
        cudaGraphExec_t exec = nullptr;
        int64_t launches = 0;           // kernels in the captured sequence
        long long last_use = 0;
    } gslot[2];
    long long gclock = 0;
    int64_t graph_replays = 0;
    float* d_static = nullptr;          // device address of g_static_scratch on this handle's device (osiv_tv_gradient_static)
    // per-kernel event timing (osiv_set_profiling)
    bool profiling = false;
    std::vector<cudaEvent_t> events;
    double prof_ms_fwd = 0.0, prof_ms_back = 0.0;
    int64_t prof_n_fwd = 0, prof_n_back = 0;
};

// ---- scratch of the allocation-free entry point (osiv_tv_gradient_static) --------------------------------------
// The padded images of that call live here instead of in cudaMalloc'ed workspace.  The array is part of the module
// image: every device that loads the library holds OSIV_STATIC_SCRATCH_BYTES of it until the process exits.  In host
// code the name below is only a stand-in for the symbol, not a device address: the address comes from
// cudaGetSymbolAddress, once per device with that device current (static_scratch_address, called by osiv_create).
static __device__ __align__(256) float g_static_scratch[OSIV_STATIC_SCRATCH_BYTES / sizeof(float)];

constexpr int STATIC_MAX_DEVICES = 64;
static float* g_static_addr[STATIC_MAX_DEVICES] = {};

// [batch][ny][nx] -> zero-bordered row-major copies (DevGeom::sb == 1), the layout k_tv reads; borders are cleared by
// the caller
__global__ void __launch_bounds__(256) k_pad_rows(DevGeom g, const float* __restrict__ src, float* __restrict__ img) {
    const int s = blockIdx.z;
    const int x = blockIdx.x * 32 + (threadIdx.x & 31);
    const int y = blockIdx.y * 8 + (threadIdx.x >> 5);
    if (x >= g.nx || y >= g.ny) return;
    img[(size_t)s * g.img_elems + pad_off(g, y, x)] = src[((size_t)s * g.ny + y) * g.nx + x];
}

namespace {

// device address of g_static_scratch on `device`, which must be current; null if the lookup fails (the entry point
// then reports OSIV_ERR_CUDA).  No allocation: the array already exists on every device that loaded the module.
float* static_scratch_address(int device) {
    if (device < 0 || device >= STATIC_MAX_DEVICES) return nullptr;
    if (!g_static_addr[device]) {
        float* p = nullptr;
        if (cudaGetSymbolAddress((void**)&p, g_static_scratch) != cudaSuccess) { cudaGetLastError(); return nullptr; }
        g_static_addr[device] = p;
    }
    return g_static_addr[device];
}

struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; prev = -1; return; }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// OSIV_DEBUG=1 in the environment names the failing CUDA call on stderr (diagnostics; the library is otherwise silent)
inline bool cuda_failed(cudaError_t e, const char* what) {
    if (e == cudaSuccess) return false;
    if (std::getenv("OSIV_DEBUG")) std::fprintf(stderr, "libosiv: %s: %s\n", what, cudaGetErrorString(e));
    cudaGetLastError();
    return true;
}
#define OSIV_CUDA(call) do { if (cuda_failed((call), #call)) return OSIV_ERR_CUDA; } while (0)

// bumped whenever a workspace buffer is (re)allocated: a captured graph holds device pointers and is dropped when this moves
long long g_alloc_gen = 0;

template <class T>
int grow(T** p, size_t* have, size_t want) {
    if (*have >= want && *p) return OSIV_OK;
    ++g_alloc_gen;
    if (*p) { OSIV_CUDA(cudaFree(*p)); *p = nullptr; *have = 0; }
    OSIV_CUDA(cudaMalloc((void**)p, want * sizeof(T)));
    *have = want;
    return OSIV_OK;
}

double resolve_dgamma(const osiv_geometry& g) {
    if (g.dgamma_rad > 0.0) return g.dgamma_rad;
    const int nmin = g.nx < g.ny ? g.nx : g.ny;
    return 2.0 * std::asin(0.5 * nmin * g.pixel_mm / g.sad_mm) / g.n_channels;
}

// A0: per-ray coefficients {alpha, beta, g0, h} in float64, stored float32 (header of osiv_kernels.cuh).
// Ray (v,c): direction d = -(cos phi, sin phi), phi = th_v + ga_c; signed distance of the point
// D*(xc,yc) from it: p = D*(xc*dy - yc*dx) + SAD*sin(ga_c).
// With V % 4 == 0 the views of the second to fourth quarter turn are written as the exact rotations
// (alpha,beta,g0,h) -> (-beta,alpha,g0,h) of the first quarter's (the same numbers up to the last bit of the
// float64 cosines), which is what lets both kernels share one weight across a quarter-turn orbit.
void build_tables(const osiv_geometry& g, double dgamma, std::vector<float4>& rays, std::vector<float2>& views) {
    const int V = g.n_views, C = g.n_channels;
    const double D = g.pixel_mm, tiny = 1e-9;
    rays.resize((size_t)V * C);
    views.resize(V);
    const int Vq = (V % 4 == 0) ? V / 4 : V;
    for (int v = 0; v < V; ++v) {
        const double th = g.theta0_rad + 2.0 * M_PI * (double)v / (double)V;
        views[v] = make_float2((float)std::cos(th), (float)std::sin(th));
        if (v >= Vq) {
            for (int c = 0; c < C; ++c) {
                const float4 q = rays[(size_t)(v - Vq) * C + c];
                rays[(size_t)v * C + c] = make_float4(-q.y, q.x, q.z, q.w);
            }
            continue;
        }
        for (int c = 0; c < C; ++c) {
            const double ga = ((double)c - 0.5 * (C - 1) + g.channel_offset) * dgamma;
            double dx = -std::cos(th + ga), dy = -std::sin(th + ga);
            const double S = g.sad_mm * std::sin(ga);
            float4 r;
            if (std::fabs(dy) >= std::fabs(dx)) {          // crosses every row once: in-line coordinate is x
                if (std::fabs(dx) < tiny) dx = dx < 0 ? -tiny : tiny;
                r.x = (float)(-dy / dx);                   // p / (-D dx)
                r.y = 1.f;
                r.z = (float)(-S / (D * dx));
                r.w = (float)(D / std::fabs(dy));
            } else {                                       // crosses every column once: in-line coordinate is y
                if (std::fabs(dy) < tiny) dy = dy < 0 ? -tiny : tiny;
                r.x = 1.f;                                 // p / (D dy)
                r.y = (float)(-dx / dy);
                r.z = (float)(S / (D * dy));
                r.w = (float)(D / std::fabs(dx));
            }
            if (g.model == 1) {
                // Joseph: a = h * sat(1 - |xc - x*|) on the ray's major-axis line, and |xc - x*| = |q| / |k| with k the
                // in-line coefficient: the same expression with the ray's three coefficients divided by |k|
                // (in-line coefficient +-1, marching coefficient +-1/|k|) and a half-width of 1
                const double ak = std::fabs(dy) >= std::fabs(dx) ? std::fabs(dy / dx) : std::fabs(dx / dy);
                if (std::fabs(dy) >= std::fabs(dx)) { r.x = (-dy / dx) > 0 ? 1.f : -1.f; r.y = (float)(1.0 / ak); r.z = (float)(-S / (D * dx) / ak); }
                else                                { r.x = (float)(1.0 / ak); r.y = (-dx / dy) > 0 ? 1.f : -1.f; r.z = (float)(S / (D * dy) / ak); }
            }
            rays[(size_t)v * C + c] = r;
        }
    }
}

int subset_views(const osiv_handle* h, int subset, int n_subsets) {
    return subset < 0 ? h->geom.n_views : h->geom.n_views / n_subsets;
}

int check_subset(const osiv_handle* h, int subset, int n_subsets) {
    if (subset < 0) return OSIV_OK;
    if (n_subsets <= 0 || h->geom.n_views % n_subsets != 0 || subset >= n_subsets) return OSIV_ERR_INVALID_ARG;
    return OSIV_OK;
}

// padded image buffers for `batch` slices in the layout (sb, ns): slices interleaved per pixel in groups of sb; ns = 1:
// one float per pixel, ns = 4: the orbit float4 per pixel (header of osiv_kernels.cuh).  The buffers are sized for the
// float4 layout when the geometry admits it; the pads are zeroed when the buffers are made or the layout changes and
// never written again.
int ensure_images(osiv_handle* h, int batch, int sb, int ns, cudaStream_t st) {
    const int slices = (batch + sb - 1) / sb * sb;
    h->dg.sb = sb;
    if (h->ws_batch >= slices && h->ws_sb == sb && h->ws_ns == ns) return OSIV_OK;
    const int n = std::max(slices, h->ws_batch);
    const size_t per = h->dg.sym4 ? 4 : 1;
    const size_t ne = (size_t)h->dg.img_elems * n * per, nt = (size_t)h->dg.imgT_elems * n * per;
    if (h->ws_batch < slices) {
        float** bufs[4] = {&h->d_imgA, &h->d_imgB, &h->d_imgTA, &h->d_imgTB};
        for (auto b : bufs) if (*b) { OSIV_CUDA(cudaFree(*b)); *b = nullptr; }
        if (h->d_best) { OSIV_CUDA(cudaFree(h->d_best)); h->d_best = nullptr; }
        h->ws_batch = 0;
        ++g_alloc_gen;
        OSIV_CUDA(cudaMalloc((void**)&h->d_imgA, ne * sizeof(float)));
        OSIV_CUDA(cudaMalloc((void**)&h->d_imgB, ne * sizeof(float)));
        OSIV_CUDA(cudaMalloc((void**)&h->d_imgTA, nt * sizeof(float)));
        OSIV_CUDA(cudaMalloc((void**)&h->d_imgTB, nt * sizeof(float)));
        OSIV_CUDA(cudaMalloc((void**)&h->d_best, (size_t)h->geom.nx * h->geom.ny * n * sizeof(float)));
    }
    OSIV_CUDA(cudaMemsetAsync(h->d_imgA, 0, ne * sizeof(float), st));
    OSIV_CUDA(cudaMemsetAsync(h->d_imgB, 0, ne * sizeof(float), st));
    OSIV_CUDA(cudaMemsetAsync(h->d_imgTA, 0, nt * sizeof(float), st));
    OSIV_CUDA(cudaMemsetAsync(h->d_imgTB, 0, nt * sizeof(float), st));
    h->ws_batch = n;
    h->ws_sb = sb;
    h->ws_ns = ns;
    return OSIV_OK;
}

// ---- launch plans -------------------------------------------------------------------------------------
// NS = 4 (quarter-turn orbits share one weight) needs a square grid with nx % 4 == 0, V % 4 == 0 and a subset
// made of whole orbits (V_S % 4 == 0); everything else takes the general NS = 1 kernels.
// A stack of slices (view_shift / tv_z) always takes the general kernels.
int pick_ns(const osiv_handle* h, int VS, bool stack = false) { return (h->dg.sym4 && !h->force_ns1 && !stack && VS % 4 == 0) ? 4 : 1; }

constexpr int BATCH_THREADS = 512;      // K1 block size cap when a launch carries several slices: two blocks per SM
constexpr int BATCH_MIN_SLICES = 4;     // fewer slices than this run one after the other in full-size blocks

// Launches with several slices serve pairs of slices per block (SB = 2: interleaved images, shared chord weights) when
// K2's tiles per block leave room for at least one view share in its 448-thread blocks.
int pick_sb(const osiv_handle* h, int VS, int batch, bool stack) {
    if (batch < BATCH_MIN_SLICES || stack) return 1;      // a stack's slices differ in their views: no pairs
    const int ns = pick_ns(h, VS, stack);
    const int tx = ns == 4 ? h->geom.nx / 4 : (h->geom.nx + BK_TX - 1) / BK_TX;
    const int ty = ns == 4 ? h->geom.ny / 4 : (h->geom.ny + BK_TY - 1) / BK_TY;
    const long long tiles = (long long)(((tx + BK_WX - 1) / BK_WX + 1) / 2) * (((ty + BK_WY - 1) / BK_WY + 1) / 2) * 4 * 32;
    const long long tpb = (std::max<long long>(1, (tiles + h->num_sms - 1) / h->num_sms) + 7) / 8 * 8;
    return tpb * ns <= BKB_MAX_THREADS ? 2 : 1;
}

struct FwdPlan { int threads, rpb, segs, nparts, ns, sb; size_t smem; };

// magic of osiv::fastdiv: n / d == umulhi(n, ceil(2^32 / d)) for 0 <= n < 2^32 / d (every use here stays below 2^21)
unsigned div_magic(int d) { return d <= 1 ? 0u : (unsigned)(((1ull << 32) + (unsigned)d - 1) / (unsigned)d); }
struct BackPlan { int nblk, threads, tpb, shares, ngx, ns, sb, ntiles; size_t smem; };

// K1: the subset's base rays are dealt out in runs of rpb consecutive rays, one run per block and one block per SM
// (per slice); a block is rpb rays x segs segments of each ray's line range, as many segments as fit into 1024
// threads while a segment keeps at least FWD_MIN_LINES image lines.
FwdPlan plan_forward(const osiv_handle* h, int VS, int batch, bool stack = false) {
    FwdPlan p;
    p.ns = pick_ns(h, VS, stack);
    const long long R = (long long)(VS / p.ns) * h->geom.n_channels;
    p.rpb = (int)std::min<long long>(FWD_MAX_THREADS, std::max<long long>(1, (R + h->num_sms - 1) / h->num_sms));
    const int nmax = std::max(h->geom.nx, h->geom.ny);
    // several slices (A8): pairs of slices share the chord weights (SB = 2), in half-size blocks, two per SM, which
    // fill each other's stalls
    p.sb = pick_sb(h, VS, batch, stack);
    const int tmax = std::max(p.rpb, p.sb == 2 ? BATCH_THREADS : FWD_MAX_THREADS);
    p.segs = std::max(1, std::min(tmax / p.rpb, nmax / FWD_MIN_LINES));
    // A thread walks its segment in trips of `lpt` lines (k_forward's LPT): the fewest segments that keep the number of trips
    // -- fewer warps to start, to meet at the barrier and to sum over; config 3: 19 x 27 lines instead of 20 x 26, seven
    // trips either way, +0.35 %; thinning 1/40: 32 x 16 instead of 40 x 13
    {
        const int lpt = (p.ns == 4 && p.sb == 1) ? 4 : 2;
        const int len = (nmax + p.segs - 1) / p.segs, trips = (len + lpt - 1) / lpt;
        p.segs = std::max(1, std::min(p.segs, (nmax + trips * lpt - 1) / (trips * lpt)));
    }
    p.threads = (p.rpb * p.segs + 31) / 32 * 32;
    p.nparts = (int)((R + p.rpb - 1) / p.rpb);
    p.smem = (size_t)p.sb * p.segs * p.ns * p.rpb * sizeof(float);
    return p;
}

template <int MODE>
cudaError_t launch_forward(FwdPlan p, int batch, const FwdArgs& a, cudaStream_t st, bool pdl) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(p.nparts, 1, (batch + p.sb - 1) / p.sb); cfg.blockDim = dim3(p.threads);
    cfg.dynamicSmemBytes = p.smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
    if (p.sb == 2) return p.ns == 4 ? cudaLaunchKernelEx(&cfg, k_forward<MODE, 4, 2>, a) : cudaLaunchKernelEx(&cfg, k_forward<MODE, 1, 2>, a);
    return p.ns == 4 ? cudaLaunchKernelEx(&cfg, k_forward<MODE, 4, 1>, a) : cudaLaunchKernelEx(&cfg, k_forward<MODE, 1, 1>, a);
}

// K2: the base tiles, numbered patch by patch (8 x 4 tiles, patches grouped 2 x 2), are dealt out in runs of tpb
// consecutive tiles, one run per block and one block per SM (per slice); a block is tpb tiles x `shares` view shares.
BackPlan plan_back(const osiv_handle* h, int VS, int batch, bool stack = false) {
    BackPlan p;
    p.ns = pick_ns(h, VS, stack);
    const int tx = p.ns == 4 ? h->geom.nx / 4 : (h->geom.nx + BK_TX - 1) / BK_TX;
    const int ty = p.ns == 4 ? h->geom.ny / 4 : (h->geom.ny + BK_TY - 1) / BK_TY;
    p.ngx = ((tx + BK_WX - 1) / BK_WX + 1) / 2;
    const int ngy = ((ty + BK_WY - 1) / BK_WY + 1) / 2;
    const long long tiles = (long long)p.ngx * ngy * 4 * 32;
    p.ntiles = (int)tiles;
    p.tpb = (int)std::min<long long>(BK_MAX_THREADS / p.ns, std::max<long long>(1, (tiles + h->num_sms - 1) / h->num_sms));
    // whole units of 8 tiles (4 x 2, the lanes of a quarter-warp: tile_origin) per block, so that every 16-byte load of the
    // candidate loop is served for 8 neighbouring tiles
    p.tpb = std::min((p.tpb + 7) / 8 * 8, BK_MAX_THREADS / p.ns / 8 * 8);
    p.nblk = (int)((tiles + p.tpb - 1) / p.tpb);
    const int VSb = VS / p.ns;
    // shares per quarter turn (NS == 4) or in all: as many as fit, then the fewest that keep the same number of
    // views per share
    // several slices: pairs of slices share the chord weights in blocks of at most 448 threads, two blocks per SM (A8)
    p.sb = pick_sb(h, VS, batch, stack);
    const int tmax = std::max(p.tpb * p.ns, p.sb == 2 ? BKB_MAX_THREADS : BK_MAX_THREADS);
    int sq = std::max(1, std::min(tmax / (p.tpb * p.ns), VSb));
    const int trips = (VSb + sq - 1) / sq;
    sq = (VSb + trips - 1) / trips;
    p.shares = sq * p.ns;
    p.threads = (p.tpb * p.shares + 31) / 32 * 32;
    p.smem = (size_t)p.sb * p.shares * p.ns * 4 * p.tpb * sizeof(float);
    return p;
}

template <int MODE>
cudaError_t launch_back(const BackPlan& p, int batch, const BackArgs& a, cudaStream_t st, bool pdl) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(p.nblk, 1, (batch + p.sb - 1) / p.sb); cfg.blockDim = dim3(p.threads); cfg.stream = st;
    cfg.dynamicSmemBytes = p.smem;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
    if (p.sb == 2) return p.ns == 4 ? cudaLaunchKernelEx(&cfg, k_back<MODE, 4, 2, 0>, a) : cudaLaunchKernelEx(&cfg, k_back<MODE, 1, 2, 0>, a);
    if (MODE == 1 && (a.view_shift != 0 || a.tv_z > 0.f)) return cudaLaunchKernelEx(&cfg, k_back<1, 1, 1, 1>, a);      // a stack: ns == 1
    return p.ns == 4 ? cudaLaunchKernelEx(&cfg, k_back<MODE, 4, 1, 0>, a) : cudaLaunchKernelEx(&cfg, k_back<MODE, 1, 1, 0>, a);
}

// ---- staged K2 (osiv_back_staged.cuh) ------------------------------------------------------------------
constexpr size_t SMEM_OPTIN = 227 * 1024;       // shared memory one block may ask for on sm_100

// The base quadrant in tiles of 4 x 2 pixels (TX x TY) is cut into nblk rectangles of about equal area: rows of blocks,
// each row cut into nb_r columns; every rectangle must hold at most BS_MAX_TPB tiles.  Returns {} when that fails.
std::vector<int4> staged_regions(int TX, int TY, int nblk, int* tpb_out) {
    std::vector<int4> out;
    int nrows = std::max(1, (int)std::lround(std::sqrt((double)nblk * (TY * (double)BS_TY) / (TX * (double)BS_TX))));
    nrows = std::min(std::min(nrows, TY), nblk);
    if ((nblk + nrows - 1) / nrows > TX) return out;
    std::vector<int> nb(nrows), hgt(nrows), wmax(nrows);
    int cum = 0, y_prev = 0;
    for (int r = 0; r < nrows; ++r) {
        nb[r] = nblk / nrows + (r < nblk % nrows ? 1 : 0);
        cum += nb[r];
        int y = (int)std::floor((double)TY * cum / nblk + 0.5);
        y = std::max(y, y_prev + 1);
        y = std::min(y, TY - (nrows - 1 - r));
        hgt[r] = y - y_prev;
        y_prev = y;
        wmax[r] = (TX + nb[r] - 1) / nb[r];
    }
    // move tile rows from block rows whose widest rectangle is too large to the block row with the most room
    for (int guard = 0; guard < 4 * TY; ++guard) {
        int bad = -1;
        for (int r = 0; r < nrows; ++r) if (wmax[r] * hgt[r] > BS_MAX_TPB && (bad < 0 || wmax[r] * hgt[r] > wmax[bad] * hgt[bad])) bad = r;
        if (bad < 0) break;
        int to = -1;
        for (int r = 0; r < nrows; ++r)
            if (r != bad && wmax[r] * (hgt[r] + 1) <= BS_MAX_TPB && (to < 0 || wmax[r] * (hgt[r] + 1) < wmax[to] * (hgt[to] + 1))) to = r;
        if (to < 0 || hgt[bad] <= 1) return out;
        hgt[bad] -= 1; hgt[to] += 1;
    }
    int tpb = 0, y0 = 0;
    for (int r = 0; r < nrows; ++r) {
        if (wmax[r] * hgt[r] > BS_MAX_TPB) { out.clear(); return out; }
        for (int k = 0; k < nb[r]; ++k) {
            const int x0 = (int)((long long)TX * k / nb[r]), x1 = (int)((long long)TX * (k + 1) / nb[r]);
            const int w = x1 - x0;
            out.push_back(make_int4(x0 | (y0 << 16), w | (hgt[r] << 16), (int)div_magic(w), 0));
            tpb = std::max(tpb, w * hgt[r]);
        }
        y0 += hgt[r];
    }
    *tpb_out = tpb;
    return out;
}

// A0 for the staged K2, at osiv_create: regions, per-(view, block) windows and per-tile candidate intervals.  Leaves
// h->st_ready = 0 (the general K2 serves) when the geometry does not qualify; an error only for CUDA failures.
int build_staged(osiv_handle* h, double tile_hw_staged) {
    const osiv_geometry& g = h->geom;
    h->st_ready = 0;
    if (!h->dg.sym4 || g.nx % (2 * BS_TX) != 0 || h->dgamma * g.n_channels >= 0.5 * M_PI) return OSIV_OK;
    const int TX = g.nx / 2 / BS_TX, TY = g.ny / 2 / BS_TY;
    const long long tiles = (long long)TX * TY;
    // whole multiples of the SM count, about 56 tiles per block; small grids: at least 8 tiles per block
    const long long tgt = 60;           // (30 or 20 tiles per block, two or three blocks per SM, measured 9 and 24 % slower)
    int nblk = (int)std::min<long long>((long long)h->num_sms * ((tiles + tgt * h->num_sms - 1) / (tgt * h->num_sms)),
                                        std::max<long long>(1, tiles / 8));
    std::vector<int4> regions;
    int tpb = 0;
    for (int tries = 0; tries < 8 && regions.empty(); ++tries, nblk += h->num_sms)
        if (nblk <= BS_MAX_REGIONS) regions = staged_regions(TX, TY, nblk, &tpb);
    if (regions.empty()) return OSIV_OK;
    nblk = (int)regions.size();
    const int tpbp = (tpb + 31) / 32 * 32;
    const size_t n_itab = (size_t)g.n_views * nblk * tpbp;
    int* d_max = nullptr;
    int hmax[2] = {0, 0};
    if (cudaMalloc((void**)&h->d_regions, regions.size() * sizeof(int4)) != cudaSuccess ||
        cudaMalloc((void**)&h->d_itab2, n_itab * sizeof(unsigned short)) != cudaSuccess ||
        cudaMalloc((void**)&h->d_bwin, (size_t)g.n_views * nblk * sizeof(int)) != cudaSuccess ||
        cudaMalloc((void**)&d_max, 2 * sizeof(int)) != cudaSuccess ||
        cudaMemset(d_max, 0, 2 * sizeof(int)) != cudaSuccess ||
        cudaMemcpy(h->d_regions, regions.data(), regions.size() * sizeof(int4), cudaMemcpyHostToDevice) != cudaSuccess) {
        if (d_max) cudaFree(d_max);
        cudaGetLastError();
        return OSIV_ERR_CUDA;
    }
    k_build_staged<<<dim3(nblk, g.n_views), tpbp>>>(h->dg, (float)tile_hw_staged, g.model == 1 ? 0.f : 0.5f, g.model == 1 ? 1.f : 0.5f,
                                                    h->d_regions, nblk, tpbp, h->d_itab2, h->d_bwin, d_max);
    h->launches += 1;
    const bool ok = cudaMemcpy(hmax, d_max, sizeof(hmax), cudaMemcpyDeviceToHost) == cudaSuccess;
    cudaFree(d_max);
    if (!ok) { cudaGetLastError(); return OSIV_ERR_CUDA; }
    // a lane walks up to the warp's largest count from its own first candidate
    const int W = (hmax[0] + hmax[1] + 1) / 2 * 2;
    if (hmax[0] >= 256 || hmax[1] >= 255 || W > 512) return OSIV_OK;
    const size_t slot = 16 + (size_t)W * 8 + (size_t)tpbp * 2 + (size_t)W * 16;       // constants + residual window
    const size_t fixed = BS_HDR_BYTES + (size_t)BS_SHARES * tpbp * BS_RED_PITCH * sizeof(float4);
    if (fixed + 4 * slot > SMEM_OPTIN || 4 > BS_RCH * ((BS_SHARES * tpbp) / W)) return OSIV_OK;
    if (cudaFuncSetAttribute(k_back_staged<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_OPTIN) != cudaSuccess ||
        cudaFuncSetAttribute(k_back_staged<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_OPTIN) != cudaSuccess) {
        cudaGetLastError();
        return OSIV_ERR_CUDA;
    }
    h->st_nblk = nblk; h->st_tpbp = tpbp; h->st_W = W;
    h->st_regions = regions;
    h->st_ready = 1;
    return OSIV_OK;
}

struct StagedPlan { int nblk, tpbp, threads, W, JR, nrounds, slot_c; size_t smem; };

// the blob of the staged K2 for M subsets (M = 1: all views in one), rebuilt when M changes
int ensure_blob(osiv_handle* h, int M, cudaStream_t st) {
    if (h->d_blob && h->blob_M == M) return OSIV_OK;
    const int V = h->geom.n_views, VS = V / M;
    const int slot_c = 16 + h->st_W * 8 + h->st_tpbp * 2;
    const size_t want = (size_t)V * h->st_nblk * slot_c;
    h->blob_M = 0;
    int rc = grow(&h->d_blob, &h->blob_bytes, want);
    if (rc != OSIV_OK) return rc;
    k_build_blob<<<dim3(h->st_nblk, VS, M), 128, 0, st>>>(h->dg, M, VS, h->st_nblk, h->st_tpbp, h->st_W, slot_c, h->d_itab2, h->d_bwin, h->d_blob);
    h->launches += 1;
    OSIV_CUDA(cudaGetLastError());
    h->blob_M = M;
    return OSIV_OK;
}

StagedPlan plan_staged(const osiv_handle* h, int VS) {
    StagedPlan p;
    p.nblk = h->st_nblk; p.tpbp = h->st_tpbp; p.W = h->st_W;
    p.threads = BS_SHARES * p.tpbp;
    p.slot_c = 16 + p.W * 8 + p.tpbp * 2;
    const size_t per_view = 4 * ((size_t)p.slot_c + (size_t)p.W * 16);
    const size_t fixed = BS_HDR_BYTES + (size_t)BS_SHARES * p.tpbp * BS_RED_PITCH * sizeof(float4);
    const int VSb = VS / 4;
    p.JR = (int)std::min<size_t>(std::min(VSb, BS_MAX_JR), (SMEM_OPTIN - fixed) / per_view);
    p.JR = std::max(1, std::min(p.JR, BS_RCH * (p.threads / p.W) / 4));       // a thread fetches at most BS_RCH residual chunks per round
    p.nrounds = (VSb + p.JR - 1) / p.JR;
    p.smem = fixed + (size_t)p.JR * per_view;
    return p;
}

// The staged K2 serves one slice per block on the quarter-turn path when the subset's windows fit its shared memory in ONE
// round (config 3: 10 base views).  With several rounds (all 800 views in osiv_backward: 13 rounds, each with its barriers
// and a fresh fetch) the general kernel is faster -- 5a 0.118 against 0.144 ms, 5b 0.90 against 1.22 ms per pass -- and takes
// those calls; osiv_set_back_kernel(h, 2) stages them anyway (tests of the round logic).
bool use_staged(const osiv_handle* h, const BackPlan& p, bool stack, int VS) {
    if (!(h->st_ready && h->st_off != 1 && p.ns == 4 && p.sb == 1 && !stack)) return false;
    return h->st_off == 2 || plan_staged(h, VS).nrounds == 1;
}
// ... and K1's monitor partials per slice fit the step-rule warp's registers
bool use_staged(const osiv_handle* h, const BackPlan& p, bool stack, int VS, const FwdPlan& f) {
    return use_staged(h, p, stack, VS) && f.nparts <= 32 * BS_DPK;
}

template <int MODE>
cudaError_t launch_back_staged(const osiv_handle* h, const StagedPlan& p, int batch, const BackArgs& a, cudaStream_t st, bool pdl) {
    BackSArgs sa;
    sa.b = a;
    sa.regions = h->d_regions; sa.blob = h->d_blob;
    sa.nblk = p.nblk; sa.tpbp = p.tpbp; sa.tpbp_magic = div_magic(p.tpbp); sa.W = p.W; sa.W_magic = div_magic(p.W); sa.SP = p.threads / p.W; sa.JR = p.JR; sa.nrounds = p.nrounds;
    sa.slot_c = p.slot_c;
    sa.hka = h->geom.model == 1 ? 0.f : 0.5f; sa.hkb = h->geom.model == 1 ? 1.f : 0.5f;
    if (p.nblk <= BS_PARAM_REGIONS) std::memcpy(sa.regions_c, h->st_regions.data(), (size_t)p.nblk * sizeof(int4));
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(p.nblk, 1, batch); cfg.blockDim = dim3(p.threads); cfg.stream = st;
    cfg.dynamicSmemBytes = p.smem;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, k_back_staged<MODE>, sa);
}

// K2's candidate intervals for this orbit size: one pass of k_build_intervals over all views, on first use
int ensure_intervals(osiv_handle* h, const BackPlan& p, cudaStream_t st) {
    const int w = p.ns == 4 ? 1 : 0;
    if (h->d_itab[w] && h->itab_tiles[w] == p.ntiles) return OSIV_OK;
    // one table at a time: the other orbit size's table (osiv_set_symmetry toggled, or a subset without whole orbits) goes
    for (int k = 0; k < 2; ++k)
        if (h->d_itab[k]) { OSIV_CUDA(cudaFree(h->d_itab[k])); h->d_itab[k] = nullptr; h->itab_tiles[k] = 0; }
    ++g_alloc_gen;
    OSIV_CUDA(cudaMalloc((void**)&h->d_itab[w], (size_t)h->geom.n_views * p.ntiles * sizeof(int)));
    k_build_intervals<<<dim3((p.ntiles + 255) / 256, h->geom.n_views), 256, 0, st>>>(h->dg, p.ns, p.ngx, div_magic(p.ngx), p.ntiles, h->d_itab[w]);
    h->itab_tiles[w] = p.ntiles;
    h->launches += 1;
    OSIV_CUDA(cudaGetLastError());
    return OSIV_OK;
}

int ensure_forward_ws(osiv_handle* h, const FwdPlan& p, int batch) {
    return grow(&h->d_dparts, &h->dpart_elems, (size_t)batch * p.nparts);
}

// K1's block line ranges for M subsets (M = 1: all views), rebuilt when M or the block shape changes
int ensure_fwd_ranges(osiv_handle* h, const FwdPlan& p, int M, cudaStream_t st) {
    const long long key = (((long long)M * 8 + p.ns) * 4096 + p.rpb) * 65536 + p.nparts;
    if (h->d_k1rng && h->k1rng_key == key) return OSIV_OK;
    h->k1rng_key = -1;
    int rc = grow(&h->d_k1rng, &h->k1rng_elems, (size_t)M * p.nparts);
    if (rc != OSIV_OK) return rc;
    k_build_fwd_ranges<<<dim3(p.nparts, M), (p.rpb + 31) / 32 * 32, 0, st>>>(h->dg, M, h->geom.n_views / M, p.ns, p.rpb, h->d_k1rng);
    h->launches += 1;
    OSIV_CUDA(cudaGetLastError());
    // the order in which K1's blocks take the runs: a block's walk is as long as the longer of its two line ranges
    h->k1order.clear();
    if (p.nparts <= FWD_ORDER_MAX) {
        std::vector<int4> rng((size_t)M * p.nparts);
        OSIV_CUDA(cudaMemcpyAsync(rng.data(), h->d_k1rng, rng.size() * sizeof(int4), cudaMemcpyDeviceToHost, st));
        OSIV_CUDA(cudaStreamSynchronize(st));
        h->k1order.resize(rng.size());
        std::vector<int> idx(p.nparts);
        for (int m = 0; m < M; ++m) {
            const int4* r = rng.data() + (size_t)m * p.nparts;
            for (int b = 0; b < p.nparts; ++b) idx[b] = b;
            auto cost = [&](int b) { return std::max(std::max(r[b].y - r[b].x + 1, r[b].w - r[b].z + 1), 0); };
            std::stable_sort(idx.begin(), idx.end(), [&](int x, int y) { return cost(x) > cost(y); });
            for (int b = 0; b < p.nparts; ++b) h->k1order[(size_t)m * p.nparts + b] = (unsigned short)idx[b];
        }
    }
    h->k1rng_key = key;
    return OSIV_OK;
}

// residual buffer [batch][V_S][Cp] floats (NS == 4: [batch][V_S/4][Cp] float4); columns C..Cp-1 must be zero, and they
// move when the layout changes, so the buffer is cleared whenever (V_S, orbit size, batch) differs from the last call
int ensure_res(osiv_handle* h, int VS, int ns, int batch, cudaStream_t st) {
    const int Cp = h->geom.n_channels + h->res_pad;
    const size_t want = (size_t)batch * VS * Cp;
    const long long key = ((long long)VS * 8 + ns) * 100000 + batch;
    const bool realloc = h->res_elems < want || !h->d_res;
    int rc = grow(&h->d_res, &h->res_elems, want);
    if (rc != OSIV_OK) return rc;
    if (realloc || key != h->res_key) {
        OSIV_CUDA(cudaMemsetAsync(h->d_res, 0, h->res_elems * sizeof(float), st));
        h->res_key = key;
    }
    return OSIV_OK;
}

dim3 px_grid(const osiv_handle* h, int batch) { return dim3((h->geom.nx + 31) / 32, (h->geom.ny + 7) / 8, batch); }

int launch_check(osiv_handle* h, int n) {
    h->launches += n;
    OSIV_CUDA(cudaGetLastError());
    return OSIV_OK;
}

}  // namespace

extern "C" {

int osiv_version(void) { return 200; }

const char* osiv_strerror(int status) {
    switch (status) {
        case OSIV_OK: return "ok";
        case OSIV_ERR_INVALID_ARG: return "invalid argument";
        case OSIV_ERR_CUDA: return "CUDA error (no usable device, out of memory or launch failure)";
        case OSIV_ERR_NOT_FINITE: return "monitor D became non-finite";
        case OSIV_ERR_SCRATCH_LIMIT: return "osiv_tv_gradient_static: batch * (ny + 2) * (nx + 8) * 4 bytes exceed OSIV_STATIC_SCRATCH_BYTES (4 MiB)";
        default: return "unknown status";
    }
}

int osiv_default_params(osiv_params* p) {
    if (!p) return OSIV_ERR_INVALID_ARG;
    std::memset(p, 0, sizeof(*p));
    p->beta = 0.005; p->n_subsets = 1; p->n_iters = 1;
    p->mu0 = 0.005;                                     // PAPER.md:140 (0.05 /cm)
    p->lambda0 = 0.01; p->lambda_up = 1e-4; p->lambda_down = 2e-4;
    p->lambda_min = 1e-4; p->kappa = 100.0; p->tv_eps = 1e-5;
    p->return_best = 0; p->monitor_mode = 0; p->view_shift = 0; p->reserved = 0; p->tv_z = 0.0; p->forced_lambda = nullptr;
    return OSIV_OK;
}

static int check_geometry(const osiv_geometry& g) {
    // n_views is a gridDim.y of the set-up kernels (k_build_intervals, k_scale_sino)
    if (g.nx <= 0 || g.ny <= 0 || g.n_views <= 0 || g.n_channels <= 0 || g.nx > 16384 || g.ny > 16384 ||
        g.n_views > 65535 || g.n_channels >= (1 << 20) ||
        (g.model != 0 && g.model != 1) || g.reserved != 0)
        return OSIV_ERR_INVALID_ARG;
    if (!(g.pixel_mm > 0.0) || !(g.sad_mm > 0.0) || !std::isfinite(g.pixel_mm) || !std::isfinite(g.sad_mm) ||
        !std::isfinite(g.dgamma_rad) || !std::isfinite(g.channel_offset) || !std::isfinite(g.theta0_rad))
        return OSIV_ERR_INVALID_ARG;
    const double rmax = 0.5 * g.pixel_mm * std::sqrt((double)g.nx * g.nx + (double)g.ny * g.ny);
    if (!(g.sad_mm > rmax * 1.0001)) return OSIV_ERR_INVALID_ARG;      // source must be outside the grid
    if (g.dgamma_rad <= 0.0 && 0.5 * (g.nx < g.ny ? g.nx : g.ny) * g.pixel_mm >= g.sad_mm) return OSIV_ERR_INVALID_ARG;
    const double dgamma = resolve_dgamma(g);
    if (!(dgamma > 0.0) || dgamma * g.n_channels >= M_PI) return OSIV_ERR_INVALID_ARG;
    return OSIV_OK;
}

int osiv_ray_table(const osiv_geometry* geom, float* h_rays, float* h_views) {
    if (!geom || check_geometry(*geom) != OSIV_OK) return OSIV_ERR_INVALID_ARG;
    std::vector<float4> rays;
    std::vector<float2> views;
    build_tables(*geom, resolve_dgamma(*geom), rays, views);
    if (h_rays) std::memcpy(h_rays, rays.data(), rays.size() * sizeof(float4));      // {alpha, beta, g0, h}
    if (h_views) std::memcpy(h_views, views.data(), views.size() * sizeof(float2));
    return OSIV_OK;
}

int osiv_create(const osiv_geometry* geom, int32_t max_batch, int32_t device, osiv_handle** out) {
    if (out) *out = nullptr;
    if (!geom || !out || max_batch <= 0 || device < 0) return OSIV_ERR_INVALID_ARG;
    const osiv_geometry& g = *geom;
    if (check_geometry(g) != OSIV_OK) return OSIV_ERR_INVALID_ARG;
    const double rmax = 0.5 * g.pixel_mm * std::sqrt((double)g.nx * g.nx + (double)g.ny * g.ny);
    const double dgamma = resolve_dgamma(g);

    DeviceGuard guard(device);
    if (!guard.ok) { cudaGetLastError(); return OSIV_ERR_CUDA; }

    osiv_handle* h = new (std::nothrow) osiv_handle();
    if (!h) return OSIV_ERR_CUDA;
    h->geom = g; h->dgamma = dgamma; h->device = device; h->max_batch = max_batch;
    h->d_static = static_scratch_address(device);     // set-up for osiv_tv_gradient_static; a failure shows there

    std::vector<float4> rays;
    std::vector<float2> views;
    build_tables(g, dgamma, rays, views);
    // K2 reads up to res_pad entries past a view's last channel: zero slack after the last view
    // rays that can have a non-zero weight for one of a tile's pixels pass within tile_r of the tile's centre: exact
    // chord -- they cross the tile's square; Joseph -- within pixel*max(|dx|,|dy|) <= pixel of a pixel centre
    const double tile_r = g.model == 1
        ? 0.5 * g.pixel_mm * std::sqrt((double)((BK_TX - 1) * (BK_TX - 1) + (BK_TY - 1) * (BK_TY - 1))) + g.pixel_mm
        : 0.5 * g.pixel_mm * std::sqrt((double)(BK_TX * BK_TX + BK_TY * BK_TY));
    const double xm = std::min(tile_r / (g.sad_mm - rmax), 1.0);
    const double tile_hw = std::asin(xm) / xm * tile_r / dgamma * 1.0005;
    h->res_pad = ((2 * (int)std::ceil(tile_hw / (g.sad_mm - rmax) + 0.05) + 3) + 3) / 4 * 4;
    // device layout: float4 {alpha, beta, g0, hk} for the inner loops, h in a table of its own
    std::vector<float> hs(rays.size());
    for (size_t i = 0; i < rays.size(); ++i) {
        hs[i] = rays[i].w;
        rays[i].w = g.model == 1 ? 1.f : 0.5f * (std::fabs(rays[i].x) + std::fabs(rays[i].y));
    }
    // zero slack after the last view: K2 reads past a view's last channel (general kernel: res_pad entries; staged
    // kernel: up to one window of at most 512 entries)
    std::vector<float> invk(rays.size());
    for (size_t i = 0; i < rays.size(); ++i) invk[i] = 1.0f / (std::fabs(rays[i].x) >= std::fabs(rays[i].y) ? rays[i].x : rays[i].y);
    rays.resize(rays.size() + h->res_pad + 4 + 512, make_float4(0.f, 0.f, 0.f, 0.f));
    h->ray_entries = (long long)rays.size();
    if (cudaMalloc((void**)&h->d_rays, rays.size() * sizeof(float4)) != cudaSuccess ||
        cudaMalloc((void**)&h->d_hs, hs.size() * sizeof(float)) != cudaSuccess ||
        cudaMemcpy(h->d_hs, hs.data(), hs.size() * sizeof(float), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMalloc((void**)&h->d_invk, invk.size() * sizeof(float)) != cudaSuccess ||
        cudaMemcpy(h->d_invk, invk.data(), invk.size() * sizeof(float), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMalloc((void**)&h->d_views, views.size() * sizeof(float2)) != cudaSuccess ||
        cudaMalloc((void**)&h->d_state, (size_t)2 * max_batch * sizeof(SliceState)) != cudaSuccess ||
        cudaMalloc((void**)&h->d_not_finite, (size_t)max_batch * sizeof(int)) != cudaSuccess ||
        cudaMalloc((void**)&h->d_inv_bref, sizeof(float)) != cudaSuccess ||
        cudaMemcpy(h->d_rays, rays.data(), rays.size() * sizeof(float4), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(h->d_views, views.data(), views.size() * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess ||
        // K2's shared-memory reduction buffer: up to 1024 threads x 16 floats
        cudaFuncSetAttribute(k_back<0, 4, 1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024) != cudaSuccess ||
        cudaFuncSetAttribute(k_back<1, 4, 1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024) != cudaSuccess ||
        cudaFuncSetAttribute(k_back<0, 4, 2, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024) != cudaSuccess ||
        cudaFuncSetAttribute(k_back<1, 4, 2, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024) != cudaSuccess) {
        cudaGetLastError();
        osiv_destroy(h);
        return OSIV_ERR_CUDA;
    }

    DevGeom& d = h->dg;
    d.nx = g.nx; d.ny = g.ny; d.V = g.n_views; d.C = g.n_channels;
    d.pitch = g.nx + 2 * PAD; d.pitchT = g.ny + 2 * PAD;
    d.img_elems = (long long)(g.ny + 2 * PADR) * d.pitch;
    d.imgT_elems = (long long)(g.nx + 2 * PADR) * d.pitchT;
    d.cx = 0.5f * (g.nx - 1); d.cy = 0.5f * (g.ny - 1);
    d.pixel = (float)g.pixel_mm; d.sad = (float)g.sad_mm;
    d.inv_dgamma = (float)(1.0 / dgamma);
    d.c_center = (float)(0.5 * (g.n_channels - 1) - g.channel_offset);
    // K2 candidate bound: every ray through a tile passes within its half-diagonal r of the tile centre, so its fan
    // angle is within asin(r/L) <= f*r/along of the centre's, f = asin(x)/x at the largest possible x = r/(SAD-r_max)
    d.tile_hw = (float)tile_hw;
    // atan_small: |z| <= 0.75, error 3e-7 rad; demand < 0.01 channel, else atanf
    const double zmax = rmax / (g.sad_mm - rmax);
    d.use_atanf = (zmax > 0.75 || 3e-7 / dgamma > 0.01) ? 1 : 0;
    d.sym4 = (g.nx == g.ny && g.nx % 4 == 0 && g.n_views % 4 == 0) ? 1 : 0;
    d.sb = 1;
    d.rays = h->d_rays; d.views = h->d_views; d.hs = h->d_hs;
    {
        // staged K2: its tiles are 4 x 2 pixels (same bound as tile_hw with that tile's radius)
        const double tr = g.model == 1
            ? 0.5 * g.pixel_mm * std::sqrt((double)((BS_TX - 1) * (BS_TX - 1) + (BS_TY - 1) * (BS_TY - 1))) + g.pixel_mm
            : 0.5 * g.pixel_mm * std::sqrt((double)(BS_TX * BS_TX + BS_TY * BS_TY));
        const double xs = std::min(tr / (g.sad_mm - rmax), 1.0);
        const int rc = build_staged(h, std::asin(xs) / xs * tr / dgamma * 1.0005);
        if (rc != OSIV_OK) { osiv_destroy(h); return rc; }
        // the staged kernel copies whole windows of a residual row: the row's zero columns must cover one window
        if (h->st_ready) h->res_pad = std::max(h->res_pad, (h->st_W + 3) / 4 * 4);
    }
    *out = h;
    return OSIV_OK;
}

int osiv_destroy(osiv_handle* h) {
    if (!h) return OSIV_OK;
    DeviceGuard guard(h->device);
    if (guard.ok) {
        cudaDeviceSynchronize();
        void* ptrs[] = {h->d_rays, h->d_views, h->d_hs, h->d_imgA, h->d_imgB, h->d_imgTA, h->d_imgTB, h->d_best, h->d_res,
                        h->d_dparts, h->d_state, h->d_not_finite, h->d_inv_bref, h->d_trace,
                        h->d_forced, h->d_dhist, h->d_itab[0], h->d_itab[1], h->d_hcounts, h->d_hblank, h->d_himg,
                        h->d_regions, h->d_itab2, h->d_bwin, h->d_blob, h->d_invk, h->d_k1rng};
        for (void* p : ptrs) if (p) cudaFree(p);
        for (cudaEvent_t e : h->events) cudaEventDestroy(e);
        for (auto& gs : h->gslot) if (gs.exec) cudaGraphExecDestroy(gs.exec);
        if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
        cudaGetLastError();
    }
    delete h;
    return OSIV_OK;
}

int osiv_get_dgamma(const osiv_handle* h, double* dgamma_rad) {
    if (!h || !dgamma_rad) return OSIV_ERR_INVALID_ARG;
    *dgamma_rad = h->dgamma;
    return OSIV_OK;
}

int osiv_get_tau(const osiv_handle* h, int32_t n_subsets, double kappa, double* tau) {
    if (!h || !tau || n_subsets <= 0 || h->geom.n_views % n_subsets != 0) return OSIV_ERR_INVALID_ARG;
    const osiv_geometry& g = h->geom;
    const int N = g.nx > g.ny ? g.nx : g.ny;
    const double vs = (double)(g.n_views / n_subsets), d = g.pixel_mm;
    *tau = kappa * g.sad_mm * h->dgamma / (vs * N * d * d * d);       // C6
    return OSIV_OK;
}

int64_t osiv_launch_count(const osiv_handle* h) { return h ? h->launches : 0; }

int osiv_debug_checks(uint64_t* h_out3) {
#ifdef OSIV_CHECKED
    if (!h_out3) return OSIV_ERR_INVALID_ARG;
    OSIV_CUDA(cudaDeviceSynchronize());
    OSIV_CUDA(cudaMemcpyFromSymbol(h_out3, g_check, 3 * sizeof(unsigned long long)));
    return OSIV_OK;
#else
    (void)h_out3;
    return OSIV_ERR_INVALID_ARG;                          // not the checked build
#endif
}

int osiv_debug_timeline(uint64_t* h_out, int32_t n_entries) {
#ifdef OSIV_TRACE
    if (!h_out || n_entries != 4 * TL_BLOCKS * TL_SLOTS) return OSIV_ERR_INVALID_ARG;
    OSIV_CUDA(cudaDeviceSynchronize());
    OSIV_CUDA(cudaMemcpyFromSymbol(h_out, g_timeline, sizeof(unsigned long long) * 4 * TL_BLOCKS * TL_SLOTS));
    return OSIV_OK;
#else
    (void)h_out; (void)n_entries;
    return OSIV_ERR_INVALID_ARG;                          // not the timeline build
#endif
}

int osiv_set_symmetry(osiv_handle* h, int32_t enable) {
    if (!h) return OSIV_ERR_INVALID_ARG;
    h->force_ns1 = enable ? 0 : 1;
    return OSIV_OK;
}

int osiv_set_back_kernel(osiv_handle* h, int32_t mode) {
    if (!h || mode < 0 || mode > 2) return OSIV_ERR_INVALID_ARG;
    h->st_off = mode;
    return OSIV_OK;
}

int osiv_set_graph(osiv_handle* h, int32_t enable) {
    if (!h) return OSIV_ERR_INVALID_ARG;
    h->use_graph = enable ? 1 : 0;
    return OSIV_OK;
}

int64_t osiv_graph_replays(const osiv_handle* h) { return h ? h->graph_replays : 0; }

int osiv_get_back_kernel(const osiv_handle* h, int32_t n_subsets, int32_t batch, int32_t* staged) {
    if (!h || !staged || batch <= 0 || (n_subsets > 0 && h->geom.n_views % n_subsets != 0)) return OSIV_ERR_INVALID_ARG;
    const int VS = n_subsets > 0 ? h->geom.n_views / n_subsets : h->geom.n_views;
    *staged = use_staged(h, plan_back(h, VS, batch), false, VS) ? 1 : 0;
    return OSIV_OK;
}

int osiv_set_overlap(osiv_handle* h, int32_t enable) {
    if (!h) return OSIV_ERR_INVALID_ARG;
    h->use_pdl = enable ? 1 : 0;
    return OSIV_OK;
}

int osiv_get_plan(const osiv_handle* h, int32_t n_subsets, int32_t batch, int32_t* out8) {
    if (!h || !out8 || batch <= 0 || (n_subsets > 0 && h->geom.n_views % n_subsets != 0)) return OSIV_ERR_INVALID_ARG;
    const int VS = n_subsets > 0 ? h->geom.n_views / n_subsets : h->geom.n_views;
    const FwdPlan f = plan_forward(h, VS, batch);
    const BackPlan b = plan_back(h, VS, batch);
    out8[0] = f.ns; out8[1] = f.segs; out8[2] = f.nparts * ((batch + f.sb - 1) / f.sb); out8[3] = f.threads;
    out8[4] = b.ns; out8[5] = b.shares; out8[6] = b.nblk * ((batch + b.sb - 1) / b.sb); out8[7] = b.threads;
    if (use_staged(h, b, false, VS)) {
        const StagedPlan sp = plan_staged(h, VS);
        out8[5] = BS_SHARES; out8[6] = sp.nblk * batch; out8[7] = sp.threads;
    }
    return OSIV_OK;
}

int osiv_set_profiling(osiv_handle* h, int32_t enable) {
    if (!h) return OSIV_ERR_INVALID_ARG;
    h->profiling = enable != 0;
    h->prof_ms_fwd = h->prof_ms_back = 0.0;
    h->prof_n_fwd = h->prof_n_back = 0;
    return OSIV_OK;
}

int osiv_get_profile(const osiv_handle* h, double* ms_forward, int64_t* n_forward, double* ms_back, int64_t* n_back) {
    if (!h) return OSIV_ERR_INVALID_ARG;
    if (ms_forward) *ms_forward = h->prof_ms_fwd;
    if (n_forward) *n_forward = h->prof_n_fwd;
    if (ms_back) *ms_back = h->prof_ms_back;
    if (n_back) *n_back = h->prof_n_back;
    return OSIV_OK;
}

int osiv_forward(osiv_handle* h, const float* d_img, float* d_sino, int32_t batch, int32_t subset,
                 int32_t n_subsets, void* cuda_stream) {
    if (!h || !d_img || !d_sino || batch <= 0 || batch > h->max_batch) return OSIV_ERR_INVALID_ARG;
    if (check_subset(h, subset, n_subsets) != OSIV_OK) return OSIV_ERR_INVALID_ARG;
    DeviceGuard guard(h->device);
    if (!guard.ok) { cudaGetLastError(); return OSIV_ERR_CUDA; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int VS = subset_views(h, subset, n_subsets);
    const FwdPlan p = plan_forward(h, VS, batch);
    int rc = ensure_images(h, batch, p.sb, p.ns, st);
    if (rc != OSIV_OK) return rc;
    if ((rc = ensure_forward_ws(h, p, batch)) != OSIV_OK) return rc;
    k_pad_transpose<<<px_grid(h, batch), 256, 0, st>>>(h->dg, p.ns, d_img, h->d_imgA, h->d_imgTA);
    FwdArgs a{};
    a.g = h->dg; a.img = h->d_imgA; a.imgT = h->d_imgTA;
    a.subset = subset; a.M = subset < 0 ? 1 : n_subsets; a.VS = VS; a.batch = batch; a.rpb = p.rpb; a.segs = p.segs; a.rpb_magic = div_magic(p.rpb); a.C_magic = div_magic(h->geom.n_channels); a.sino = d_sino;
    if ((rc = ensure_fwd_ranges(h, p, a.M, st)) != OSIV_OK) return rc;
    a.rng_tab = h->d_k1rng; a.invk = h->d_invk; a.segs_magic = div_magic(p.segs);
    if (launch_forward<0>(p, batch, a, st, false) != cudaSuccess) { cudaGetLastError(); return OSIV_ERR_CUDA; }
    return launch_check(h, 2);
}

int osiv_backward(osiv_handle* h, const float* d_sino, float* d_img, int32_t batch, int32_t subset,
                  int32_t n_subsets, void* cuda_stream) {
    if (!h || !d_img || !d_sino || batch <= 0 || batch > h->max_batch) return OSIV_ERR_INVALID_ARG;
    if (check_subset(h, subset, n_subsets) != OSIV_OK) return OSIV_ERR_INVALID_ARG;
    DeviceGuard guard(h->device);
    if (!guard.ok) { cudaGetLastError(); return OSIV_ERR_CUDA; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int VS = subset_views(h, subset, n_subsets), M = subset < 0 ? 1 : n_subsets;
    const BackPlan p = plan_back(h, VS, batch);
    int rc = ensure_res(h, VS, p.ns, batch, st);
    if (rc != OSIV_OK) return rc;
    const int Cp = h->geom.n_channels + h->res_pad;
    k_scale_sino<<<dim3((h->geom.n_channels + 255) / 256, VS, batch), 256, 0, st>>>(h->dg, d_sino, h->d_res, subset, M, VS,
                                                                                    p.ns, Cp);
    BackArgs b{};
    b.res_floats = (long long)h->res_elems; b.ray_entries = h->ray_entries;
    b.g = h->dg; b.res = h->d_res; b.Cp = Cp; b.subset = subset; b.M = M; b.VS = VS; b.batch = batch; b.out = d_img; b.tpb = p.tpb; b.shares = p.shares; b.ngx = p.ngx; b.tpb_magic = div_magic(p.tpb); b.ngx_magic = div_magic(p.ngx);
    if (use_staged(h, p, false, VS)) {
        if ((rc = ensure_blob(h, M, st)) != OSIV_OK) return rc;
        if (launch_back_staged<0>(h, plan_staged(h, VS), batch, b, st, false) != cudaSuccess) { cudaGetLastError(); return OSIV_ERR_CUDA; }
        return launch_check(h, 2);
    }
    if ((rc = ensure_intervals(h, p, st)) != OSIV_OK) return rc;
    b.itab = h->d_itab[p.ns == 4]; b.ntiles = p.ntiles;
    if (launch_back<0>(p, batch, b, st, false) != cudaSuccess) { cudaGetLastError(); return OSIV_ERR_CUDA; }
    return launch_check(h, 2);
}

int osiv_tv_gradient(osiv_handle* h, const float* d_img, float* d_grad, int32_t batch, double tv_eps,
                     void* cuda_stream) {
    if (!h || !d_img || !d_grad || batch <= 0 || batch > h->max_batch || !(tv_eps > 0.0)) return OSIV_ERR_INVALID_ARG;
    DeviceGuard guard(h->device);
    if (!guard.ok) { cudaGetLastError(); return OSIV_ERR_CUDA; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = ensure_images(h, batch, 1, 1, st);
    if (rc != OSIV_OK) return rc;
    k_pad_transpose<<<px_grid(h, batch), 256, 0, st>>>(h->dg, 1, d_img, h->d_imgA, h->d_imgTA);
    k_tv<<<dim3((h->geom.nx + 31) / 32, (h->geom.ny + 15) / 16, batch), 128, 0, st>>>(h->dg, h->d_imgA,
                                                                                     (float)(tv_eps * tv_eps), d_grad);
    return launch_check(h, 2);
}

// Allocation-free variant of osiv_tv_gradient: the padded images go to g_static_scratch.  Only a memset and two kernel
// launches are enqueued; the handle's workspace is neither read nor grown.
int osiv_tv_gradient_static(osiv_handle* h, const float* d_img, float* d_grad, int32_t batch, double tv_eps,
                            void* cuda_stream) {
    if (!h || !d_img || !d_grad || batch <= 0 || batch > h->max_batch || !(tv_eps > 0.0)) return OSIV_ERR_INVALID_ARG;
    const size_t need = (size_t)batch * (size_t)h->dg.img_elems * sizeof(float);
    if (need > (size_t)OSIV_STATIC_SCRATCH_BYTES) return OSIV_ERR_SCRATCH_LIMIT;
    if (!h->d_static) return OSIV_ERR_CUDA;             // cudaGetSymbolAddress failed at osiv_create
    DeviceGuard guard(h->device);
    if (!guard.ok) { cudaGetLastError(); return OSIV_ERR_CUDA; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    DevGeom g = h->dg;
    g.sb = 1;
    // the array keeps the previous call's images (possibly of another geometry): clear the part this call reads
    OSIV_CUDA(cudaMemsetAsync(h->d_static, 0, need, st));
    k_pad_rows<<<px_grid(h, batch), 256, 0, st>>>(g, d_img, h->d_static);
    k_tv<<<dim3((h->geom.nx + 31) / 32, (h->geom.ny + 15) / 16, batch), 128, 0, st>>>(g, h->d_static,
                                                                                     (float)(tv_eps * tv_eps), d_grad);
    return launch_check(h, 2);
}

int osiv_reconstruct(osiv_handle* h, const float* d_counts, const float* d_blank, float blank_scalar,
                     const osiv_params* prm, int32_t batch, float* d_img_out, double* h_trace, void* cuda_stream) {
    if (!h || !d_counts || !prm || !d_img_out || batch <= 0 || batch > h->max_batch) return OSIV_ERR_INVALID_ARG;
    const int M = prm->n_subsets, N = prm->n_iters;
    if (M <= 0 || N < 0 || h->geom.n_views % M != 0 || (prm->monitor_mode != 0 && prm->monitor_mode != 1)) return OSIV_ERR_INVALID_ARG;
    if (!d_blank && !(blank_scalar > 0.f)) return OSIV_ERR_INVALID_ARG;
    if (!(prm->tv_eps > 0.0) || !std::isfinite(prm->beta) || !std::isfinite(prm->mu0) || !(prm->kappa > 0.0))
        return OSIV_ERR_INVALID_ARG;
    const bool stack = prm->view_shift != 0 || prm->tv_z > 0.0;
    if (prm->reserved != 0 || !(prm->tv_z >= 0.0) || !std::isfinite(prm->tv_z) ||
        (stack && (prm->return_best || prm->forced_lambda)))
        return OSIV_ERR_INVALID_ARG;
    if ((long long)h->geom.n_views * batch >= (1ll << 31)) return OSIV_ERR_INVALID_ARG;     // view_shift * slice stays in 32 bits
    const int vshift = (int)(((long long)prm->view_shift % h->geom.n_views + h->geom.n_views) % h->geom.n_views);
    DeviceGuard guard(h->device);
    if (!guard.ok) { cudaGetLastError(); return OSIV_ERR_CUDA; }
    cudaStream_t st = (cudaStream_t)cuda_stream;

    const int VS = h->geom.n_views / M, C = h->geom.n_channels;
    const FwdPlan fp = plan_forward(h, VS, batch, stack);
    int rc = ensure_images(h, batch, fp.sb, fp.ns, st);
    if (rc != OSIV_OK) return rc;
    const BackPlan bp = plan_back(h, VS, batch, stack);
    if ((rc = ensure_res(h, VS, fp.ns, batch, st)) != OSIV_OK) return rc;
    const int Cp = C + h->res_pad;
    if ((rc = ensure_forward_ws(h, fp, batch)) != OSIV_OK) return rc;
    if (h_trace && N > 0 && (rc = grow(&h->d_trace, &h->trace_elems, (size_t)batch * N * 2)) != OSIV_OK) return rc;
    if (prm->forced_lambda && N > 0) {
        if ((rc = grow(&h->d_forced, &h->forced_elems, (size_t)N)) != OSIV_OK) return rc;
        OSIV_CUDA(cudaMemcpyAsync(h->d_forced, prm->forced_lambda, (size_t)N * sizeof(double), cudaMemcpyHostToDevice, st));
    }
    if (prm->monitor_mode && (rc = grow(&h->d_dhist, &h->dhist_elems, (size_t)batch * 2 * M)) != OSIV_OK) return rc;
    double tau;
    osiv_get_tau(h, M, prm->kappa, &tau);

    float* best = prm->return_best ? h->d_best : nullptr;
    SliceState* state[2] = {h->d_state, h->d_state + h->max_batch};

    FwdArgs f{};
    f.g = h->dg; f.M = M; f.VS = VS; f.batch = batch; f.view_shift = vshift; f.rpb = fp.rpb; f.segs = fp.segs; f.rpb_magic = div_magic(fp.rpb); f.C_magic = div_magic(C);
    f.counts = d_counts; f.blank = d_blank; f.blank_scalar = blank_scalar; f.inv_bref = h->d_inv_bref;
    f.res = h->d_res; f.Cp = Cp; f.dparts = h->d_dparts; f.res_floats = (long long)h->res_elems;
    f.segs_magic = div_magic(fp.segs); f.invk = h->d_invk;
    if (!stack) {                                        // a stack's slices see shifted views: its blocks work their ranges out
        if ((rc = ensure_fwd_ranges(h, fp, M, st)) != OSIV_OK) return rc;
        f.rng_tab = h->d_k1rng;
    }
    BackArgs b{};
    b.res_floats = (long long)h->res_elems; b.ray_entries = h->ray_entries;
    b.g = h->dg; b.res = h->d_res; b.Cp = Cp; b.M = M; b.VS = VS; b.batch = batch; b.view_shift = vshift; b.tv_z = (float)prm->tv_z; b.best = best; b.tpb = bp.tpb; b.shares = bp.shares; b.ngx = bp.ngx; b.tpb_magic = div_magic(bp.tpb); b.ngx_magic = div_magic(bp.ngx);
    const bool staged = use_staged(h, bp, stack, VS, fp);
    const StagedPlan sp = staged ? plan_staged(h, VS) : StagedPlan{};
    if (staged) {
        if ((rc = ensure_blob(h, M, st)) != OSIV_OK) return rc;
    } else {
        if ((rc = ensure_intervals(h, bp, st)) != OSIV_OK) return rc;
        b.itab = h->d_itab[bp.ns == 4]; b.ntiles = bp.ntiles;
    }
    b.dparts = h->d_dparts; b.nparts = fp.nparts; b.not_finite = h->d_not_finite;
    b.ip.lambda0 = prm->lambda0; b.ip.up = prm->lambda_up; b.ip.down = prm->lambda_down; b.ip.lmin = prm->lambda_min;
    b.ip.forced = (prm->forced_lambda && N > 0) ? h->d_forced : nullptr;
    b.ip.trace = (h_trace && N > 0) ? h->d_trace : nullptr;
    b.ip.n_iters = N; b.ip.return_best = prm->return_best;
    b.ip.monitor_mode = prm->monitor_mode; b.ip.M = M; b.ip.dhist = h->d_dhist;
    b.tau = tau; b.beta_over_M = (float)(prm->beta / M); b.eps2 = (float)(prm->tv_eps * prm->tv_eps);

    const bool prof = h->profiling && N > 0;
    const bool pdl = h->use_pdl != 0;
    // ---- the launch sequence of the call: set-up, N x (K1, K2), the final monitor, the result.  Either enqueued on the
    // caller's stream launch by launch, or captured once into a CUDA graph (on the handle's own stream; programmatic
    // dependent launches become programmatic graph edges) and replayed with one cudaGraphLaunch while the arguments repeat.
    auto enqueue = [&](cudaStream_t st, bool prof) -> int {
    float *cur = h->d_imgA, *curT = h->d_imgTA, *nxt = h->d_imgB, *nxtT = h->d_imgTB;
    k_init_state<<<1, 32, 0, st>>>(state[0], h->d_not_finite, batch, prm->lambda0, d_blank, blank_scalar, C, h->d_inv_bref);
    k_fill<<<px_grid(h, batch), 256, 0, st>>>(h->dg, fp.ns, (float)prm->mu0, h->d_imgA, h->d_imgTA, best);
    h->launches += 2;
    if (prof) {
        while (h->events.size() < (size_t)2 * N + 1) {
            cudaEvent_t e;
            OSIV_CUDA(cudaEventCreate(&e));
            h->events.push_back(e);
        }
        OSIV_CUDA(cudaEventRecord(h->events[0], st));
    }
    for (int n = 0; n < N; ++n) {
        const int m = n % M;                               // PAPER.md:118, C11
        f.img = cur; f.imgT = curT; f.subset = m; f.iter = n; b.iter = n;
        f.use_order = (!stack && !h->k1order.empty()) ? 1 : 0;     // longest walks first: 58.16 -> 58.28 k iterations/s (shortest first: 57.95 k)
        if (f.use_order) std::memcpy(f.order, &h->k1order[(size_t)m * fp.nparts], (size_t)fp.nparts * sizeof(unsigned short));
        OSIV_CUDA(launch_forward<1>(fp, batch, f, st, pdl));
        if (prof) cudaEventRecord(h->events[2 * n + 1], st);
        b.img = cur; b.img_new = nxt; b.imgT_new = nxtT; b.subset = m;
        b.state_in = state[n & 1]; b.state_out = state[(n + 1) & 1];
        OSIV_CUDA(staged ? launch_back_staged<1>(h, sp, batch, b, st, pdl) : launch_back<1>(bp, batch, b, st, pdl));
        if (prof) cudaEventRecord(h->events[2 * n + 2], st);
        h->launches += 2;
        float* t;
        t = cur; cur = nxt; nxt = t;
        t = curT; curT = nxtT; nxtT = t;
    }
    if (prof) {
        OSIV_CUDA(cudaStreamSynchronize(st));
        for (int n = 0; n < N; ++n) {
            float a = 0.f, c = 0.f;
            OSIV_CUDA(cudaEventElapsedTime(&a, h->events[2 * n], h->events[2 * n + 1]));
            OSIV_CUDA(cudaEventElapsedTime(&c, h->events[2 * n + 1], h->events[2 * n + 2]));
            h->prof_ms_fwd += a; h->prof_ms_back += c;
        }
        h->prof_n_fwd += N; h->prof_n_back += N;
    }
    SliceState* fin = state[N & 1];
    if (prm->return_best) {
        // the final iterate competes too, judged on the subset that would come next (C12)
        f.img = cur; f.imgT = curT; f.subset = N % M; f.use_order = 0;
        if (launch_forward<1>(fp, batch, f, st, false) != cudaSuccess) { cudaGetLastError(); return OSIV_ERR_CUDA; }
        k_final_monitor<<<batch, 32, 0, st>>>(h->d_dparts, fp.nparts, fin, h->d_not_finite);
        h->launches += 2;
    }
    k_unpad<<<px_grid(h, batch), 256, 0, st>>>(h->dg, fp.ns, cur, best, fin, d_img_out);
    return launch_check(h, 1);
    };  // enqueue

    // the graph's key: everything the captured launches depend on
    struct Key {
        const void *counts, *blank, *out;
        float blank_scalar;
        int batch, has_trace, pdl, st_off, ns1;
        long long gen;
        osiv_params prm;
    } key;
    std::memset(&key, 0, sizeof(key));
    key.counts = d_counts; key.blank = d_blank; key.out = d_img_out; key.blank_scalar = blank_scalar; key.batch = batch;
    key.has_trace = h_trace != nullptr; key.pdl = h->use_pdl; key.st_off = h->st_off; key.ns1 = h->force_ns1; key.gen = g_alloc_gen;
    std::memcpy(&key.prm, prm, sizeof(osiv_params));
    const bool graphable = h->use_graph && !prof && N > 0 && !prm->forced_lambda;
    osiv_handle::GraphSlot* slot = nullptr;
    for (auto& gs : h->gslot)
        if (gs.key.size() == sizeof(key) && std::memcmp(gs.key.data(), &key, sizeof(key)) == 0) slot = &gs;
    if (!graphable) {
        if ((rc = enqueue(st, prof)) != OSIV_OK) return rc;
    } else if (!slot) {
        // a first call with these arguments is enqueued launch by launch: capturing and instantiating a thousand nodes costs
        // more than one enqueue, so the graph is built only when the arguments repeat; they take the older slot
        osiv_handle::GraphSlot& v = h->gslot[0].last_use <= h->gslot[1].last_use ? h->gslot[0] : h->gslot[1];
        if (v.exec) { cudaGraphExecDestroy(v.exec); v.exec = nullptr; }
        v.key.assign(reinterpret_cast<unsigned char*>(&key), reinterpret_cast<unsigned char*>(&key) + sizeof(key));
        v.last_use = ++h->gclock;
        if ((rc = enqueue(st, false)) != OSIV_OK) return rc;
    } else {
        slot->last_use = ++h->gclock;
        if (!slot->exec) {
            if (!h->cap_stream) OSIV_CUDA(cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking));
            const int64_t before = h->launches;
            cudaGraph_t graph = nullptr;
            bool ok = cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
            if (ok) {
                const int erc = enqueue(h->cap_stream, false);
                ok = cudaStreamEndCapture(h->cap_stream, &graph) == cudaSuccess && erc == OSIV_OK && graph;
            }
            slot->launches = h->launches - before;
            h->launches = before;
            if (ok) ok = cudaGraphInstantiate(&slot->exec, graph, 0) == cudaSuccess;
            if (graph) cudaGraphDestroy(graph);
            if (!ok) {                                    // this driver cannot capture the sequence: launch by launch from now on
                cudaGetLastError();
                slot->exec = nullptr;
                h->use_graph = 0;
                if ((rc = enqueue(st, false)) != OSIV_OK) return rc;
            }
        }
        if (slot->exec) {
            OSIV_CUDA(cudaGraphLaunch(slot->exec, st));
            h->launches += slot->launches;
            h->graph_replays += 1;
        }
    }

    if (h_trace) {
        std::vector<int> nf(batch);
        if (N > 0)
            OSIV_CUDA(cudaMemcpyAsync(h_trace, h->d_trace, (size_t)batch * N * 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
        OSIV_CUDA(cudaMemcpyAsync(nf.data(), h->d_not_finite, (size_t)batch * sizeof(int), cudaMemcpyDeviceToHost, st));
        OSIV_CUDA(cudaStreamSynchronize(st));
        for (int s = 0; s < batch; ++s) if (nf[s]) return OSIV_ERR_NOT_FINITE;
    }
    return OSIV_OK;
}

int osiv_reconstruct_host(osiv_handle* h, const float* h_counts, const float* h_blank, float blank_scalar,
                          const osiv_params* prm, int32_t batch, float* h_img_out, double* h_trace, void* cuda_stream) {
    if (!h || !h_counts || !prm || !h_img_out || batch <= 0 || batch > h->max_batch) return OSIV_ERR_INVALID_ARG;
    DeviceGuard guard(h->device);
    if (!guard.ok) { cudaGetLastError(); return OSIV_ERR_CUDA; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t nc = (size_t)batch * h->geom.n_views * h->geom.n_channels;
    const size_t ni = (size_t)batch * h->geom.nx * h->geom.ny;
    int rc;
    if ((rc = grow(&h->d_hcounts, &h->hc_elems, nc)) != OSIV_OK) return rc;
    if ((rc = grow(&h->d_himg, &h->hi_elems, ni)) != OSIV_OK) return rc;
    if (h_blank && !h->d_hblank) OSIV_CUDA(cudaMalloc((void**)&h->d_hblank, (size_t)h->geom.n_channels * sizeof(float)));
    OSIV_CUDA(cudaMemcpyAsync(h->d_hcounts, h_counts, nc * sizeof(float), cudaMemcpyHostToDevice, st));
    if (h_blank)
        OSIV_CUDA(cudaMemcpyAsync(h->d_hblank, h_blank, (size_t)h->geom.n_channels * sizeof(float), cudaMemcpyHostToDevice, st));
    rc = osiv_reconstruct(h, h->d_hcounts, h_blank ? h->d_hblank : nullptr, blank_scalar, prm, batch, h->d_himg, h_trace, st);
    if (rc != OSIV_OK && rc != OSIV_ERR_NOT_FINITE) return rc;
    // this call synchronises anyway: the sticky non-finite flags come back with the image, trace or not
    std::vector<int> nf(batch, 0);
    OSIV_CUDA(cudaMemcpyAsync(h_img_out, h->d_himg, ni * sizeof(float), cudaMemcpyDeviceToHost, st));
    OSIV_CUDA(cudaMemcpyAsync(nf.data(), h->d_not_finite, (size_t)batch * sizeof(int), cudaMemcpyDeviceToHost, st));
    OSIV_CUDA(cudaStreamSynchronize(st));
    for (int s = 0; s < batch; ++s) if (nf[s]) return OSIV_ERR_NOT_FINITE;
    return rc;
}

}  // extern "C"
