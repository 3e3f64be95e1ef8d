// dr_api.cu -- host side of libdr: the C ABI of include/dr.h (handle, workspace carving, PT constants of
// Eq. 14-21, iteration loop with periodic residual check, six-load-case bookkeeping).
// Every field update, residual and average of the method runs in the kernels of dr_kernels_*.cuh; there is no CPU fallback.
// Host arithmetic is limited to scalars: the PT constants of Eq. 14-21 (make_pt), and, for the coded kernels, the <= 256-entry
// derived tables of a launch (lambda = K - 2G/3, (theta/h) E, c^2/(theta h) R: launch_coded), formed from table values the
// kernels k_code_tables / k_pal_values produced.
#include <cuda_runtime.h>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <string>
#include <algorithm>
#include <mutex>
#include <vector>

#include "../../include/dr.h"
#include "dr_layout.cuh"
#include "dr_kernels_aux.cuh"
#include "dr_kernels_split.cuh"
#include "dr_kernels_fused.cuh"
#include "dr_kernels_tma.cuh"
#include "dr_kernels_tb2.cuh"

#ifndef FUSED_TX
#define FUSED_TX 32
#define FUSED_TY 16
#endif

struct dr_handle {
    DrLayout L;
    double h;
    cudaStream_t st;
    // workspace carving (device)
    double* buf[2][F_COUNT];
    double *K0, *G0, *K, *G;
    double* partial;            // DR_AVG_BLOCKS * 6
    double* avg_dev;            // 6
    unsigned long long* res_bits;
    unsigned long long* hmax_bits;
    unsigned char* ids;         // uint8 phase ids, tile-blocked (palette path)
    unsigned long long *palK, *palG;   // palette keys (bit patterns), 256 each
    double* pal;                // palette values K[256], G[256] after the void clamp
    bool has_pal;               // the image has at most 256 distinct (K,G) pairs
    int use_pal;                // DR_PALETTE
    unsigned int* flags;
    // host
    double* pinned;             // 64 doubles, page-locked: [0..5] averages, [8] residual, [9..14] averages at a check; dr_solve_all: [16..21] residuals, [24..59] averages
    cudaEvent_t e0, e1;
    // parameters
    double cfl, st_factor, void_rel, stag_tol;
    int ncheck, gavg, bc_mode, kernel, form;
    int device;                 // CUDA device of the workspace and the stream (every entry point switches to it)
    int stop_reason;            // dr_stop: which rule ended the last dr_solve
    double void_applied;        // void_rel currently baked into K,G
    double hmax;
    // state
    int cur;                    // ping-pong buffer that holds the current fields
    bool stress_stale;          // DR_FORM 1 with the fused kernel: stresses not yet formed from the displacement
    bool have_fields;
    int cur_lc;
    double cur_eps0;
    // results
    double Ccol[7][6];          // Ccol[lc][m] = <sigma_m> / eps0 of load case lc; row 6: the triaxial test of App. A.3
    bool have[7];
    double avg[6];
    bool have_avg;
    int iters;
    double residual, ms;
    long long launches;
    int fused_lz;
    CUtensorMap tm_state[2][F_COUNT];   // TMA descriptors of the padded boxes (both ping-pong buffers)
    CUtensorMap tm_K, tm_G;
    // stencil-coded path (DR_KERNEL 3 / 4, dr_kernels_tb2.cuh)
    unsigned long long* codes;  // [nz+5][gy2][gx2][TB2_TY][TB2_TX]
    unsigned long long *ekeys, *rkeys;   // edge-modulus and 1/H_node tables (bit patterns), 256 each
    double* tabs;               // TB2_TAB_N table values
    double tabs_host[TB2_TAB_N];   // host copy (the derived tables of a launch are formed from it, TB2_CTAB)
    bool has_codes;             // codes and tables are valid for (code_gavg, code_void)
    bool codes_failed;          // more than 256 distinct edge / node values for that setting: one-sweep kernel instead
    int code_gavg; double code_void;
    int tb2_lz;
    bool lz_user;               // DR_ZCHUNK set by the caller
    CUtensorMap tm2_state[2][F_COUNT];   // boxes TB2_TX x TB2_TY x 1
    // six-load-case batch (dr_solve_all): state set q belongs to load case q; set 0 is the single-solve state above
    int nsets;                  // 6 if the workspace holds six state sets (dr_workspace_bytes_six), else 1
    double* xbuf[TB2_NLC][2][F_COUNT];
    CUtensorMap xtm2[TB2_NLC][2][F_COUNT];
    double* partial6;           // [6][DR_AVG_BLOCKS][6]
    double* avg6_dev;           // [6][6]
    int lc_iters[6], lc_stop[6];
    double lc_res[6];
    std::string err;
};

static dr_status fail(dr_handle* H, dr_status s, const std::string& msg) {
    if (H) H->err = msg;
    return s;
}

static bool cuda_ok(dr_handle* H, cudaError_t e, const char* what) {
    if (e == cudaSuccess) return true;
    if (H) H->err = std::string(what) + ": " + cudaGetErrorString(e);
    return false;
}

// every entry point runs on the device the handle was created on and restores the caller's device on return
struct DrDeviceGuard {
    int prev; bool sw;
    explicit DrDeviceGuard(int dev) : prev(-1), sw(false) {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) sw = (cudaSetDevice(dev) == cudaSuccess);
    }
    ~DrDeviceGuard() { if (sw) cudaSetDevice(prev); }
};

#define CK(call) do { if (!cuda_ok(H, (call), #call)) return DR_ERR_CUDA; } while (0)
#define CKL(what) do { H->launches++; if (!cuda_ok(H, cudaGetLastError(), what)) return DR_ERR_CUDA; } while (0)

static size_t align_up(size_t a, size_t m) { return (a + m - 1) / m * m; }

static bool sizes_ok(int nx, int ny, int nz) {
    return nx >= 2 && ny >= 2 && nz >= 2 && nx <= 8192 && ny <= 8192 && nz <= 8192;
}

static size_t field_bytes(const DrLayout& L) { return align_up((size_t)L.count * sizeof(double), 256); }
static const int N_BIG = 2 * F_COUNT + 4;        // 18 state fields + K0, G0, K, G
static const size_t SMALL_BYTES = align_up((size_t)DR_AVG_BLOCKS * 6 * sizeof(double), 256) + 1024 + 3 * 4096;   // + palette keys and values
static int tiles_x(const DrLayout& L) { return (L.nx + 1 + FUSED_TX - 3) / (FUSED_TX - 2); }
static int tiles_y(const DrLayout& L) { return (L.ny + 1 + FUSED_TY - 3) / (FUSED_TY - 2); }
// tile-blocked phase ids: one FUSED_TX*FUSED_TY byte block per (tile, layer), layers -1 .. nz+1
static size_t ids_bytes(const DrLayout& L) { return align_up((size_t)tiles_x(L) * tiles_y(L) * (L.nz + 3) * (FUSED_TX * FUSED_TY), 256); }

static int tb2_tiles_x(const DrLayout& L) { return (L.nx + 2 + TB2_TX - 5) / (TB2_TX - 4); }     // owned columns start at i = -1
static int tb2_tiles_y(const DrLayout& L) { return (L.ny + 1 + TB2_TY - 5) / (TB2_TY - 4); }
// stencil codes: one 8-byte word per (tile, layer, thread), layers -TB2_KLO .. nz-1+TB2_KHI; + tables and their keys
static size_t codes_bytes(const DrLayout& L) {
    return align_up((size_t)tb2_tiles_x(L) * tb2_tiles_y(L) * (L.nz + TB2_KLO + TB2_KHI) * (TB2_TX * TB2_TY) * sizeof(unsigned long long), 256);
}
static const size_t CODE_SMALL_BYTES = 2 * 2048 + TB2_TAB_N * sizeof(double);

extern "C" size_t dr_workspace_bytes(int nx, int ny, int nz) {
    if (!sizes_ok(nx, ny, nz)) return 0;
    DrLayout L = dr_make_layout(nx, ny, nz);
    return (size_t)N_BIG * field_bytes(L) + ids_bytes(L) + SMALL_BYTES + codes_bytes(L) + CODE_SMALL_BYTES;
}

// five more state sets (2 x 9 fields each) and the reduction scratch of six simultaneous load cases
static const size_t SIX_SMALL_BYTES = align_up((size_t)6 * DR_AVG_BLOCKS * 6 * sizeof(double), 256) + 512;
extern "C" size_t dr_workspace_bytes_six(int nx, int ny, int nz) {
    if (!sizes_ok(nx, ny, nz)) return 0;
    DrLayout L = dr_make_layout(nx, ny, nz);
    return dr_workspace_bytes(nx, ny, nz) + (size_t)5 * 2 * F_COUNT * field_bytes(L) + SIX_SMALL_BYTES;
}

// z-chunk length of the fused kernels: make the CTA count fill whole waves of 148 SMs while keeping the priming
// overhead (one extra step per chunk) small.  Chunks are capped at DR_LZ_MAX layers (and may be as short as 1-3 layers on tiny grids, where filling the 148 SMs matters more than the priming step): measured on B200, CTAs of
// neighbouring tiles drift apart on longer marches and the halo rows/columns they share stop hitting in L2
// (479^3: 3.53 ms/iteration at 24-32 layers per chunk, 3.67 at 48, 4.37 at 64, 5.2 at 96).
#define DR_LZ_MAX 36
#define DR_LZ_FIXED 3      // per-CTA start-up (barrier init, first TMA round trip) in units of one z step
static int choose_lz_for(int tiles, int layers, int priming, int lz_max) {
    int best_lz = layers < lz_max ? layers : lz_max;
    double best = 1e300;
    for (int lz = 1; lz <= lz_max && lz <= layers; ++lz) {
        const int chunks = (layers + lz - 1) / lz;
        const double waves = std::ceil((double)tiles * chunks / 148.0);
        const double cost = waves * (lz + priming + DR_LZ_FIXED);          // steps on the critical path of one SM
        if (cost < best - 1e-9 || (cost < best + 1e-9 && lz > best_lz)) { best = cost; best_lz = lz; }
    }
    return best_lz;
}
static int choose_lz(const DrLayout& L) {
    return choose_lz_for(tiles_x(L) * tiles_y(L), L.nz + 1, 1, DR_LZ_MAX);
}
// the two-iteration kernel runs lz + 4 steps per chunk (two priming steps per iteration); it is not DRAM-bound, so longer
// marches cost nothing in halo reuse (479^3: 2.57 ms per iteration at 32 layers, 2.52 at 60, flat beyond)
#define DR_LZ_MAX_TB2 64
static int choose_lz_tb2(const DrLayout& L) {
    return choose_lz_for(tb2_tiles_x(L) * tb2_tiles_y(L), L.nz + 1, 4, DR_LZ_MAX_TB2);
}

// TMA descriptor of one padded field: 3-D fp64 tensor (PX,PY,PZ), box (FUSED_TX, FUSED_TY, 1), no swizzle,
// out-of-range elements read as zero.  cuTensorMapEncodeTiled is fetched through the runtime (no -lcuda).
typedef CUresult (*dr_encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static bool make_tmap(dr_handle* H, dr_encode_fn enc, CUtensorMap* out, double* base, int bx = FUSED_TX, int by = FUSED_TY) {
    const DrLayout& L = H->L;
    cuuint64_t dims[3] = {(cuuint64_t)L.PX, (cuuint64_t)L.PY, (cuuint64_t)L.PZ};
    cuuint64_t strides[2] = {(cuuint64_t)L.PX * 8, (cuuint64_t)L.PX * L.PY * 8};
    cuuint32_t box[3] = {(cuuint32_t)bx, (cuuint32_t)by, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    const CUtensorMapL2promotion promo = CU_TENSOR_MAP_L2_PROMOTION_NONE;   // 64/128/256 B measured: no difference
    CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     CU_TENSOR_MAP_SWIZZLE_NONE, promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { H->err = "cuTensorMapEncodeTiled failed (" + std::to_string((int)r) + ")"; return false; }
    return true;
}

static bool make_all_tmaps(dr_handle* H) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess || !fn) {
        H->err = "cudaGetDriverEntryPoint(cuTensorMapEncodeTiled) failed";
        return false;
    }
    dr_encode_fn enc = (dr_encode_fn)fn;
    for (int b = 0; b < 2; ++b) for (int f = 0; f < F_COUNT; ++f) if (!make_tmap(H, enc, &H->tm_state[b][f], H->buf[b][f])) return false;
    for (int b = 0; b < 2; ++b) for (int f = 0; f < F_COUNT; ++f) if (!make_tmap(H, enc, &H->tm2_state[b][f], H->buf[b][f], TB2_TX, TB2_TY)) return false;
    for (int b = 0; b < 2; ++b) for (int f = 0; f < F_COUNT; ++f) H->xtm2[0][b][f] = H->tm2_state[b][f];
    for (int q = 1; q < H->nsets; ++q) for (int b = 0; b < 2; ++b) for (int f = 0; f < F_COUNT; ++f)
        if (!make_tmap(H, enc, &H->xtm2[q][b][f], H->xbuf[q][b][f], TB2_TX, TB2_TY)) return false;
    return make_tmap(H, enc, &H->tm_K, H->K) && make_tmap(H, enc, &H->tm_G, H->G);
}

// page-locked scratch of a handle (64 doubles: residuals and averages read back at a check).  cudaMallocHost / cudaFreeHost
// cost more than a whole PT iteration on small grids (the free synchronises the device), so blocks are recycled through a
// process-wide free list and live until the process ends.
static std::mutex g_pin_mu;
static std::vector<double*> g_pin_free;
static double* pinned_acquire() {
    {
        std::lock_guard<std::mutex> lk(g_pin_mu);
        if (!g_pin_free.empty()) { double* p = g_pin_free.back(); g_pin_free.pop_back(); return p; }
    }
    double* p = nullptr;
    if (cudaHostAlloc((void**)&p, 64 * sizeof(double), cudaHostAllocPortable) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return p;
}
static void pinned_release(double* p) {
    if (!p) return;
    std::lock_guard<std::mutex> lk(g_pin_mu);
    g_pin_free.push_back(p);
}

// opt in to the large dynamic shared memory of the fused kernels (all instantiations), once per device and process: the
// ~30 attribute calls are a visible part of dr_create on small grids
static cudaError_t set_kernel_attributes(int device) {
    static bool done[64] = {false};
    static std::mutex mu;                       // dr_create may be called from several host threads
    std::lock_guard<std::mutex> lk(mu);
    if (device >= 0 && device < 64 && done[device]) return cudaSuccess;
    const cudaFuncAttribute A = cudaFuncAttributeMaxDynamicSharedMemorySize;
    const int smem = (int)DrFusedCfg<FUSED_TX, FUSED_TY>::SMEM;
    cudaError_t e = cudaFuncSetAttribute(k_pt_fused<0, 0, FUSED_TX, FUSED_TY>, A, smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pt_fused<0, 1, FUSED_TX, FUSED_TY>, A, smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pt_fused<1, 0, FUSED_TX, FUSED_TY>, A, smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pt_fused<1, 1, FUSED_TX, FUSED_TY>, A, smem);
    const int smem_t = (int)DrTmaCfg2<FUSED_TX, FUSED_TY, 0>::SMEM2, smem_p = (int)DrTmaCfg2<FUSED_TX, FUSED_TY, 1>::SMEM2;
#define DR_SET_TMA_ATTR(G_, R_, F_) if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pt_tma<G_, R_, F_, 0, FUSED_TX, FUSED_TY>, A, smem_t); \
                                    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pt_tma<G_, R_, F_, 1, FUSED_TX, FUSED_TY>, A, smem_p)
    DR_SET_TMA_ATTR(0, 0, 0); DR_SET_TMA_ATTR(0, 1, 0); DR_SET_TMA_ATTR(1, 0, 0); DR_SET_TMA_ATTR(1, 1, 0);
    DR_SET_TMA_ATTR(0, 0, 1); DR_SET_TMA_ATTR(0, 1, 1); DR_SET_TMA_ATTR(1, 0, 1); DR_SET_TMA_ATTR(1, 1, 1);
#undef DR_SET_TMA_ATTR
    const int smem2 = (int)DrTb2Cfg<TB2_TX, TB2_TY>::SMEM;
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pt_tb2<0, 2, TB2_TX, TB2_TY>, A, smem2);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pt_tb2<1, 2, TB2_TX, TB2_TY>, A, smem2);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pt_tb2<0, 1, TB2_TX, TB2_TY>, A, smem2);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pt_tb2<1, 1, TB2_TX, TB2_TY>, A, smem2);
    if (e == cudaSuccess && device >= 0 && device < 64) done[device] = true;
    return e;
}

// dr_create and dr_create_segmented: the moduli come from dense fp64 arrays (K, G) or from phase ids + host tables
static dr_status create_impl(int nx, int ny, int nz, double h, const double* K, const double* G,
                             const unsigned char* phase, int nphase, const double* K_table, const double* G_table,
                             void* workspace, size_t workspace_bytes, void* cuda_stream, dr_handle** out) {
    if (!out) return DR_ERR_ARG;
    *out = nullptr;
    if (!sizes_ok(nx, ny, nz) || !(h > 0.0) || !std::isfinite(h)) return DR_ERR_ARG;
    if (phase ? (nphase < 1 || nphase > 256 || !K_table || !G_table) : (!K || !G)) return DR_ERR_ARG;
    if (!workspace || ((uintptr_t)workspace & 255u) || workspace_bytes < dr_workspace_bytes(nx, ny, nz)) return DR_ERR_WORKSPACE;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return DR_ERR_CUDA; }

    dr_handle* H = new dr_handle();
    H->L = dr_make_layout(nx, ny, nz);
    H->h = h;
    H->st = (cudaStream_t)cuda_stream;
    const size_t fb = field_bytes(H->L);
    char* p = (char*)workspace;
    for (int b = 0; b < 2; ++b) for (int f = 0; f < F_COUNT; ++f) { H->buf[b][f] = (double*)p; p += fb; }
    H->K0 = (double*)p; p += fb; H->G0 = (double*)p; p += fb; H->K = (double*)p; p += fb; H->G = (double*)p; p += fb;
    H->partial = (double*)p; p += align_up((size_t)DR_AVG_BLOCKS * 6 * sizeof(double), 256);
    H->avg_dev = (double*)p; p += 256;
    H->res_bits = (unsigned long long*)p; p += 256;
    H->hmax_bits = (unsigned long long*)p; p += 256;
    H->flags = (unsigned int*)p; p += 256;
    H->palK = (unsigned long long*)p; p += 2048; H->palG = (unsigned long long*)p; p += 2048;
    H->pal = (double*)p; p += 4096;
    p = (char*)align_up((size_t)p, 256);
    H->ids = (unsigned char*)p; p += ids_bytes(H->L);
    H->codes = (unsigned long long*)p; p += codes_bytes(H->L);
    H->ekeys = (unsigned long long*)p; p += 2048; H->rkeys = (unsigned long long*)p; p += 2048;
    H->tabs = (double*)p; p += TB2_TAB_N * sizeof(double);
    for (int b = 0; b < 2; ++b) for (int f = 0; f < F_COUNT; ++f) H->xbuf[0][b][f] = H->buf[b][f];
    H->nsets = workspace_bytes >= dr_workspace_bytes_six(nx, ny, nz) ? 6 : 1;
    H->partial6 = nullptr; H->avg6_dev = nullptr;
    if (H->nsets == 6) {
        p = (char*)align_up((size_t)p, 256);
        for (int q = 1; q < 6; ++q) for (int b = 0; b < 2; ++b) for (int f = 0; f < F_COUNT; ++f) { H->xbuf[q][b][f] = (double*)p; p += fb; }
        H->partial6 = (double*)p; p += align_up((size_t)6 * DR_AVG_BLOCKS * 6 * sizeof(double), 256);
        H->avg6_dev = (double*)p; p += 512;
    }
    for (int q = 0; q < 6; ++q) { H->lc_iters[q] = 0; H->lc_stop[q] = DR_STOP_NONE; H->lc_res[q] = 0.0; }
    H->has_codes = false; H->codes_failed = false; H->code_gavg = -1; H->code_void = -1.0;
    H->tb2_lz = choose_lz_tb2(H->L); H->lz_user = false;
    H->has_pal = false; H->use_pal = 1;
    H->pinned = nullptr; H->e0 = H->e1 = nullptr;
    if (cudaGetDevice(&H->device) != cudaSuccess) { cudaGetLastError(); delete H; return DR_ERR_CUDA; }
    H->stag_tol = 1e-10; H->stop_reason = DR_STOP_NONE;
    H->cfl = 0.55; H->st_factor = 1.0; H->void_rel = 0.0; H->ncheck = 50; H->gavg = 0; H->bc_mode = 0; H->kernel = 3; H->form = 0;
    H->void_applied = 0.0; H->hmax = 0.0;
    H->cur = 0; H->have_fields = false; H->cur_lc = -1; H->cur_eps0 = 0.0;
    for (int a = 0; a < 7; ++a) { H->have[a] = false; for (int b = 0; b < 6; ++b) H->Ccol[a][b] = 0.0; }
    for (int a = 0; a < 6; ++a) H->avg[a] = 0;
    H->have_avg = false; H->iters = 0; H->residual = 0.0; H->ms = 0.0; H->launches = 0;
    H->fused_lz = choose_lz(H->L);

    dr_status st = DR_OK;
    do {
        H->pinned = pinned_acquire();
        if (!H->pinned) { H->err = "cudaHostAlloc failed"; st = DR_ERR_CUDA; break; }
        if (!cuda_ok(H, cudaEventCreate(&H->e0), "cudaEventCreate") || !cuda_ok(H, cudaEventCreate(&H->e1), "cudaEventCreate")) { st = DR_ERR_CUDA; break; }
        // state fields and moduli boxes start as zeros (halo nodes are never written afterwards)
        if (!cuda_ok(H, cudaMemsetAsync(workspace, 0, H->nsets == 6 ? dr_workspace_bytes_six(nx, ny, nz) : dr_workspace_bytes(nx, ny, nz), H->st), "cudaMemsetAsync")) { st = DR_ERR_CUDA; break; }
        if (!cuda_ok(H, cudaMemsetAsync(H->palK, 0xff, 4096, H->st), "cudaMemsetAsync")) { st = DR_ERR_CUDA; break; }     // palK and palG := EMPTY
        DrModSrc src;
        src.K = K; src.G = G; src.ids = phase; src.tab = nullptr; src.nphase = nphase;
        if (phase) {
            // the caller's tables go to the (not yet used) table block of the coded path: K at 0, G at 256
            double host_tab[512];
            for (int e = 0; e < 256; ++e) { host_tab[e] = e < nphase ? K_table[e] : 0.0; host_tab[256 + e] = e < nphase ? G_table[e] : 0.0; }
            if (!cuda_ok(H, cudaMemcpyAsync(H->tabs, host_tab, sizeof(host_tab), cudaMemcpyHostToDevice, H->st), "cudaMemcpyAsync(tables)") ||
                !cuda_ok(H, cudaStreamSynchronize(H->st), "cudaStreamSynchronize")) { st = DR_ERR_CUDA; break; }      // host_tab is a stack buffer
            src.tab = H->tabs;
        }
        dim3 blk(64, 4, 1), grd((nx + 2 + 63) / 64, (ny + 2 + 3) / 4, nz + 2);
        k_pad_moduli<<<grd, blk, 0, H->st>>>(H->L, src, H->K0, H->G0, H->flags, H->hmax_bits);
        H->launches++;
        if (!cuda_ok(H, cudaGetLastError(), "k_pad_moduli")) { st = DR_ERR_CUDA; break; }
        const long long cnt = H->L.count;
        k_void_clamp<<<(unsigned)((cnt + 255) / 256), 256, 0, H->st>>>(H->L, H->K0, H->G0, H->K, H->G, 0.0);
        H->launches++;
        if (!cuda_ok(H, cudaGetLastError(), "k_void_clamp")) { st = DR_ERR_CUDA; break; }
        // palette of the distinct (K,G) pairs; more than 256 of them (flag 2) simply leaves the fp64 path in charge
        {
            const long long Ncell = (long long)nx * ny * nz;
            k_pal_build<<<(unsigned)((Ncell + 255) / 256), 256, 0, H->st>>>(Ncell, src, H->palK, H->palG, H->flags);
            H->launches++;
            if (!cuda_ok(H, cudaGetLastError(), "k_pal_build")) { st = DR_ERR_CUDA; break; }
        }
        unsigned long long hb = 0; unsigned int fl = 0;
        if (!cuda_ok(H, cudaMemcpyAsync(&hb, H->hmax_bits, 8, cudaMemcpyDeviceToHost, H->st), "memcpy") ||
            !cuda_ok(H, cudaMemcpyAsync(&fl, H->flags, 4, cudaMemcpyDeviceToHost, H->st), "memcpy") ||
            !cuda_ok(H, cudaStreamSynchronize(H->st), "cudaStreamSynchronize")) { st = DR_ERR_CUDA; break; }
        if (fl & 1u) { st = DR_ERR_ARG; break; }
        if (!(fl & 2u)) {
            k_pal_assign<<<dim3(tiles_x(H->L), tiles_y(H->L), nz + 3), dim3(FUSED_TX, FUSED_TY, 1), 0, H->st>>>(H->L, src, H->palK, H->palG, H->ids, H->flags);
            k_pal_values<<<1, 256, 0, H->st>>>(H->palK, H->palG, H->pal, 0.0);
            H->launches += 2;
            unsigned int fl2 = 0;
            if (!cuda_ok(H, cudaGetLastError(), "k_pal_assign") ||
                !cuda_ok(H, cudaMemcpyAsync(&fl2, H->flags, 4, cudaMemcpyDeviceToHost, H->st), "memcpy") ||
                !cuda_ok(H, cudaStreamSynchronize(H->st), "cudaStreamSynchronize")) { st = DR_ERR_CUDA; break; }
            H->has_pal = !(fl2 & 4u);
        }
        std::memcpy(&H->hmax, &hb, 8);
        if (!cuda_ok(H, set_kernel_attributes(H->device), "cudaFuncSetAttribute")) { st = DR_ERR_CUDA; break; }
        if (!make_all_tmaps(H)) { st = DR_ERR_CUDA; break; }
    } while (0);
    if (st != DR_OK) {
        pinned_release(H->pinned);
        if (H->e0) cudaEventDestroy(H->e0);
        if (H->e1) cudaEventDestroy(H->e1);
        delete H;
        return st;
    }
    *out = H;
    return DR_OK;
}

extern "C" dr_status dr_create(int nx, int ny, int nz, double h, const double* K, const double* G,
                               void* workspace, size_t workspace_bytes, void* cuda_stream, dr_handle** out) {
    return create_impl(nx, ny, nz, h, K, G, nullptr, 0, nullptr, nullptr, workspace, workspace_bytes, cuda_stream, out);
}

extern "C" dr_status dr_create_segmented(int nx, int ny, int nz, double h, const unsigned char* phase, int nphase,
                                         const double* K_table, const double* G_table,
                                         void* workspace, size_t workspace_bytes, void* cuda_stream, dr_handle** out) {
    if (!phase) return DR_ERR_ARG;
    return create_impl(nx, ny, nz, h, nullptr, nullptr, phase, nphase, K_table, G_table, workspace, workspace_bytes, cuda_stream, out);
}

extern "C" dr_status dr_set_param(dr_handle* H, int id, double v) {
    if (!H) return DR_ERR_ARG;
    // parameters that shape the iterate invalidate the current fields: dr_iterate / dr_get_field then need a new
    // dr_step / dr_solve (DR_ERR_STATE) instead of silently continuing on state built under the old value
    switch (id) {
        case DR_CFL:       if (!(v > 0.0)) break; H->cfl = v; H->have_fields = false; return DR_OK;
        case DR_ST_FACTOR: if (!(v > 0.0)) break; H->st_factor = v; H->have_fields = false; return DR_OK;
        case DR_NCHECK:    if (!(v >= 1.0)) break; H->ncheck = (int)v; return DR_OK;
        case DR_GAVG:      if (v != 0.0 && v != 1.0) break; H->gavg = (int)v; H->have_fields = false; return DR_OK;
        case DR_VOID_REL:  if (!(v >= 0.0)) break; H->void_rel = v; H->have_fields = false; return DR_OK;
        case DR_BC_MODE:   if (v != 0.0 && v != 1.0) break; H->bc_mode = (int)v; H->have_fields = false; return DR_OK;
        case DR_KERNEL:    if (v != 0.0 && v != 1.0 && v != 2.0 && v != 3.0 && v != 4.0) break; H->kernel = (int)v; H->have_fields = false; return DR_OK;
        // choosing a form also resets C~ to that form's default (the explicit damping of the displacement form
        // diverges at 0.55 on small grids)
        case DR_FORM:      if (v != 0.0 && v != 1.0) break; H->form = (int)v; H->cfl = H->form ? 0.50 : 0.55; H->have_fields = false; return DR_OK;
        case DR_PALETTE:   if (v != 0.0 && v != 1.0) break; H->use_pal = (int)v; return DR_OK;
        case DR_ZCHUNK:    if (!(v >= 0.0) || v > 8192.0) break;
                           H->fused_lz = v >= 1.0 ? (int)v : choose_lz(H->L); H->tb2_lz = v >= 1.0 ? (int)v : choose_lz_tb2(H->L);
                           H->lz_user = v >= 1.0; return DR_OK;
        case DR_STAG_TOL:  if (!(v >= 0.0)) break; H->stag_tol = v; return DR_OK;
        default: break;
    }
    return fail(H, DR_ERR_ARG, "bad parameter id or value");
}

// Eq. 14-21, SURVEY O1 and O4
static DrPT make_pt(const dr_handle* H, int lc, double eps0) {
    DrPT P;
    const DrLayout& L = H->L;
    const int nmax = std::max(L.nx, std::max(L.ny, L.nz));
    const double St = 2.0 * M_PI * std::sqrt(3.0) * H->st_factor;        // St_opt in 3-D
    P.theta = H->cfl * St / nmax;                                         // dt~/Dt, from Eq. 14 and 16
    P.rinv = 1.0 / (1.0 + P.theta);
    P.c2t = H->cfl * H->cfl * H->h * H->h / P.theta;                      // Eq. 17
    P.h = H->h; P.inv_h = 1.0 / H->h;
    for (int a = 0; a < 9; ++a) P.D[a] = 0.0;
    static const int slot[6] = {0, 4, 8, 5, 2, 1};                        // Dxx Dyy Dzz Dyz Dxz Dxy
    if (lc == 6) { P.D[0] = eps0; P.D[4] = eps0; P.D[8] = eps0; }         // 7th direct test (App. A.3): triaxial
    else P.D[slot[lc]] = eps0;
    P.Lx = L.nx * H->h; P.Ly = L.ny * H->h; P.Lz = L.nz * H->h;
    P.res_scale = H->h / std::fabs(eps0);
    P.ghost_yz = (H->bc_mode == 1 || lc == 3);
    P.ghost_xz = (H->bc_mode == 1 || lc == 4);
    P.ghost_xy = (H->bc_mode == 1 || lc == 5);
    return P;
}

static DrFields fields_of(dr_handle* H, int b) {
    DrFields F; for (int f = 0; f < F_COUNT; ++f) F.f[f] = H->buf[b][f]; return F;
}
static DrConstFields cfields_of(dr_handle* H, int b) {
    DrConstFields F; for (int f = 0; f < F_COUNT; ++f) F.f[f] = H->buf[b][f]; return F;
}

// stencil codes and tables of the coded path (dr_kernels_tb2.cuh) for the current DR_GAVG / DR_VOID_REL; an image with
// more than 256 distinct (K,G) pairs, edge moduli or node stiffnesses is left uncoded (has_codes = false) and DR_KERNEL 3
// then runs the one-sweep kernel
static dr_status ensure_codes(dr_handle* H) {
    // palette off: the codes are dropped, and so is their cache key -- switching DR_PALETTE back on must rebuild them instead
    // of meeting the key below with has_codes still false (which left the handle on the one-sweep kernel)
    if (!(H->has_pal && H->use_pal)) { H->has_codes = false; H->code_gavg = -1; return DR_OK; }
    if (H->code_gavg == H->gavg && H->code_void == H->void_applied) return DR_OK;      // built (or failed) for this setting
    const DrLayout& L = H->L;
    H->has_codes = false; H->codes_failed = false;
    CK(cudaMemsetAsync(H->ekeys, 0xff, 4096, H->st));                                // ekeys and rkeys := EMPTY
    CK(cudaMemsetAsync(H->flags, 0, 4, H->st));
    dim3 blk(TB2_TX, TB2_TY, 1), grd(tb2_tiles_x(L), tb2_tiles_y(L), L.nz + TB2_KLO + TB2_KHI);
#define DR_CODE(G_, P_) k_code_build<G_, P_><<<grd, blk, 0, H->st>>>(H->L, H->K, H->G, H->K0, H->G0, H->palK, H->palG, H->ekeys, H->rkeys, H->codes, H->flags)
    if (H->gavg) DR_CODE(1, 0); else DR_CODE(0, 0);
    CKL("k_code_build<0>");
    unsigned int fl = 0;
    CK(cudaMemcpyAsync(&fl, H->flags, 4, cudaMemcpyDeviceToHost, H->st));
    CK(cudaStreamSynchronize(H->st));
    H->code_gavg = H->gavg; H->code_void = H->void_applied;
    if (fl & 8u) { H->codes_failed = true; return DR_OK; }
    if (H->gavg) DR_CODE(1, 1); else DR_CODE(0, 1);
    CKL("k_code_build<1>");
#undef DR_CODE
    k_code_tables<<<1, 256, 0, H->st>>>(H->pal, H->ekeys, H->rkeys, H->tabs);
    CKL("k_code_tables");
    CK(cudaMemcpyAsync(H->tabs_host, H->tabs, TB2_TAB_N * sizeof(double), cudaMemcpyDeviceToHost, H->st));
    CK(cudaMemcpyAsync(&fl, H->flags, 4, cudaMemcpyDeviceToHost, H->st));
    CK(cudaStreamSynchronize(H->st));
    if (fl & 16u) return fail(H, DR_ERR_CUDA, "stencil code lookup missed a table entry (internal error)");
    H->has_codes = true;
    return DR_OK;
}

// moduli-side preparation of a solve: the void clamp and, for the coded kernels, the stencil codes
static dr_status prepare_moduli(dr_handle* H) {
    const DrLayout& L = H->L;
    if (H->void_applied != H->void_rel) {
        k_void_clamp<<<(unsigned)((L.count + 255) / 256), 256, 0, H->st>>>(H->L, H->K0, H->G0, H->K, H->G, H->void_rel * H->hmax);
        CKL("k_void_clamp");
        if (H->has_pal) { k_pal_values<<<1, 256, 0, H->st>>>(H->palK, H->palG, H->pal, H->void_rel * H->hmax); CKL("k_pal_values"); }
        H->void_applied = H->void_rel;
    }
    if (H->kernel >= 3 && H->form == 0) {          // the displacement form runs the one-sweep TMA kernel
        dr_status cs = ensure_codes(H);
        if (cs != DR_OK) return cs;
    }
    return DR_OK;
}

static dr_status prepare(dr_handle* H, int lc, double eps0) {
    const DrLayout& L = H->L;
    { dr_status ms = prepare_moduli(H); if (ms != DR_OK) return ms; }
    DrPT P = make_pt(H, lc, eps0);
    dim3 blk(32, 4, 1), grd(((L.nx + 3) / 2 + 31) / 32, (L.ny + 1 + 3) / 4, (L.nz + 1 + DR_BC_ZB - 1) / DR_BC_ZB);   // pairs (2t-1, 2t), t = 0 .. (nx+2)/2
    if (H->form == 1 && H->kernel == 2) return fail(H, DR_ERR_ARG, "DR_FORM = 1 is implemented by DR_KERNEL 0 and 1 only");
    if (H->gavg) k_bc_init<1><<<grd, blk, 0, H->st>>>(H->L, P, fields_of(H, 0), fields_of(H, 1), H->form, H->K, H->G);
    else         k_bc_init<0><<<grd, blk, 0, H->st>>>(H->L, P, fields_of(H, 0), fields_of(H, 1), H->form, H->K, H->G);
    CKL("k_bc_init");
    H->cur = 0; H->have_fields = true; H->cur_lc = lc; H->cur_eps0 = eps0; H->stress_stale = false;
    return DR_OK;
}

// the coded kernels (DR_KERNEL 3, 4) need the stencil codes; without them the one-sweep TMA kernel runs
static bool coded(const dr_handle* H) { return H->kernel >= 3 && H->has_codes && H->form == 0; }

// slot `slot` of a batch launch <- state set `set` (old state in its buffer `cur`, new state into the other one)
static void fill_slot(dr_handle* H, DrTb2Batch& TB, int slot, int set, int cur, const DrPT& P) {
    static const int order[9] = {F_VX, F_VY, F_VZ, F_SXX, F_SYY, F_SZZ, F_TXY, F_TXZ, F_TYZ};
    for (int f = 0; f < 9; ++f) TB.m[slot][f] = H->xtm2[set][cur][order[f]];
    TB.out[slot] = H->xbuf[set][cur ^ 1][0];
    TB.res[slot] = H->res_bits + set;
    TB.P[slot] = P;
}

// launch the coded kernel on the first nslots slots of TB: nit PT iterations per sweep; with_res: residual of the last
static dr_status launch_coded(dr_handle* H, DrTb2Batch& TB, int nslots, bool with_res, int nit) {
    const DrLayout& L = H->L;
    // a batch of load cases multiplies the CTA count: pick the z chunk that fills whole waves for THIS number of slots
    // (small grids: 32^3 runs 2-layer chunks alone and 9-layer chunks with six load cases; results do not depend on it)
    const int lz = (H->lz_user || nslots == 1) ? H->tb2_lz
                                               : choose_lz_for(tb2_tiles_x(L) * tb2_tiles_y(L) * nslots, L.nz + 1, 4, DR_LZ_MAX_TB2);
    const int nchunks = (L.nz + 1 + lz - 1) / lz;
    dim3 blk(TB2_TX, TB2_TY, 1), grd(tb2_tiles_x(L), tb2_tiles_y(L), nchunks * nslots);
    TB.fs = H->buf[0][1] - H->buf[0][0];
    TB.codes = H->codes; TB.tabs = H->tabs; TB.gx = (int)grd.x; TB.gy = (int)grd.y; TB.nchunks = nchunks;
    TB.l2_hint = 0x1000000000000000ull;
#if TB2_CTAB
    {
        // derived tables (TB2_S_*): the same expressions, in the same order, the kernel used to evaluate per CTA; theta, h and
        // C~ are those of the handle, hence equal for every slot of a batch
        const DrPT& P0 = TB.P[0];
        const double thh = P0.theta * P0.inv_h, cvh = P0.c2t * P0.inv_h;
        for (int e = 0; e < 256; ++e) {
            const double Kv = H->tabs_host[TB2_TAB_K + e], Gv = H->tabs_host[TB2_TAB_G + e], Rv = H->tabs_host[TB2_TAB_R + e];
            TB.dtab[TB2_S_LAM + e] = std::fma(-(2.0 / 3.0), Gv, Kv);
            TB.dtab[TB2_S_G2 + e] = 2.0 * Gv;
            TB.dtab[TB2_S_ES + e] = thh * H->tabs_host[TB2_TAB_E + e];
            TB.dtab[TB2_S_CV + e] = cvh * Rv;
            TB.dtab[TB2_S_RH + e] = Rv;
        }
    }
#endif
    const size_t smem = DrTb2Cfg<TB2_TX, TB2_TY>::SMEM;
    if (nit == 2) { if (with_res) k_pt_tb2<1, 2, TB2_TX, TB2_TY><<<grd, blk, smem, H->st>>>(TB, H->L, lz);
                    else          k_pt_tb2<0, 2, TB2_TX, TB2_TY><<<grd, blk, smem, H->st>>>(TB, H->L, lz); }
    else          { if (with_res) k_pt_tb2<1, 1, TB2_TX, TB2_TY><<<grd, blk, smem, H->st>>>(TB, H->L, lz);
                    else          k_pt_tb2<0, 1, TB2_TX, TB2_TY><<<grd, blk, smem, H->st>>>(TB, H->L, lz); }
    CKL("k_pt_tb2");
    return DR_OK;
}

// nit PT iterations in one sweep of the coded kernel (dr_kernels_tb2.cuh); with_res: residual of the LAST of them
static dr_status iteration_coded(dr_handle* H, const DrPT& P, bool with_res, int nit) {
    static thread_local DrTb2Batch TB;
    fill_slot(H, TB, 0, 0, H->cur, P);
    dr_status s = launch_coded(H, TB, 1, with_res, nit);
    if (s != DR_OK) return s;
    H->cur ^= 1;
    return DR_OK;
}

// one PT iteration; with_res: also accumulate the residual max-norm into res_bits (caller zeroes it)
static dr_status iteration(dr_handle* H, const DrPT& P, bool with_res) {
    const DrLayout& L = H->L;
    if (coded(H)) return iteration_coded(H, P, with_res, 1);  // DR_KERNEL 4, and the odd single sweeps of DR_KERNEL 3
    const int kernel = H->kernel >= 3 ? 0 : H->kernel;      // uncoded images and the displacement form: the TMA kernel
    if (kernel == 1) {
        dim3 blk(64, 4, 1), grd((L.nx + 1 + 63) / 64, (L.ny + 1 + 3) / 4, L.nz + 1);
        // FORM 0: in place in buffer cur.  FORM 1: u, w in buffer cur, stresses of this iteration in buffer cur^1.
        DrFields U = fields_of(H, H->cur);
        DrFields S = fields_of(H, H->form ? H->cur ^ 1 : H->cur);
        DrConstFields Uc = cfields_of(H, H->cur), Sc = cfields_of(H, H->form ? H->cur ^ 1 : H->cur);
        dim3 grv((L.nx + 63) / 64, (L.ny + 3) / 4, L.nz);
#define DR_SPLIT(G_, F_) do { \
            k_stress_split<G_, F_><<<grd, blk, 0, H->st>>>(H->L, P, Uc, S, H->K, H->G); CKL("k_stress_split"); \
            if (with_res) k_velocity_split<G_, 1, F_><<<grv, blk, 0, H->st>>>(H->L, P, U, Sc, H->K, H->G, H->res_bits); \
            else          k_velocity_split<G_, 0, F_><<<grv, blk, 0, H->st>>>(H->L, P, U, Sc, H->K, H->G, H->res_bits); } while (0)
        if (H->gavg) { if (H->form) DR_SPLIT(1, 1); else DR_SPLIT(1, 0); }
        else         { if (H->form) DR_SPLIT(0, 1); else DR_SPLIT(0, 0); }
#undef DR_SPLIT
        CKL("k_velocity_split");
        return DR_OK;
    }
    const int lz = H->fused_lz;
    dim3 blk(FUSED_TX, FUSED_TY, 1);
    dim3 grd((L.nx + 1 + FUSED_TX - 3) / (FUSED_TX - 2), (L.ny + 1 + FUSED_TY - 3) / (FUSED_TY - 2), (L.nz + 1 + lz - 1) / lz);
    if (kernel == 0) {
        DrTmaps T;
        const int c = H->cur;
        T.m[0] = H->tm_state[c][F_VX]; T.m[1] = H->tm_state[c][F_VY]; T.m[2] = H->tm_state[c][F_VZ]; T.m[3] = H->tm_G;
        T.m[4] = H->tm_K; T.m[5] = H->tm_state[c][F_SXX]; T.m[6] = H->tm_state[c][F_SYY]; T.m[7] = H->tm_state[c][F_SZZ];
        T.m[8] = H->tm_state[c][F_TXY]; T.m[9] = H->tm_state[c][F_TXZ]; T.m[10] = H->tm_state[c][F_TYZ];
        T.l2_hint = 0x1000000000000000ull;      // L2 evict_normal (evict_first measured 20 % slower, evict_last no gain)
        const bool palp = H->has_pal && H->use_pal;          // phase-id path: same values through a 256-entry table
        T.ids = H->ids; T.pal = H->pal; T.gx = (int)grd.x; T.gy = (int)grd.y;
        const size_t smem_t = palp ? DrTmaCfg2<FUSED_TX, FUSED_TY, 1>::SMEM2 : DrTmaCfg2<FUSED_TX, FUSED_TY, 0>::SMEM2;
        DrFields Bo = fields_of(H, c ^ 1);
#define DR_TMA(G_, R_, F_) do { if (palp) k_pt_tma<G_, R_, F_, 1, FUSED_TX, FUSED_TY><<<grd, blk, smem_t, H->st>>>(T, H->L, P, Bo, lz, H->res_bits); \
                                else      k_pt_tma<G_, R_, F_, 0, FUSED_TX, FUSED_TY><<<grd, blk, smem_t, H->st>>>(T, H->L, P, Bo, lz, H->res_bits); } while (0)
        const int sel = (H->gavg ? 4 : 0) | (with_res ? 2 : 0) | (H->form ? 1 : 0);
        switch (sel) {
            case 0: DR_TMA(0, 0, 0); break; case 1: DR_TMA(0, 0, 1); break; case 2: DR_TMA(0, 1, 0); break; case 3: DR_TMA(0, 1, 1); break;
            case 4: DR_TMA(1, 0, 0); break; case 5: DR_TMA(1, 0, 1); break; case 6: DR_TMA(1, 1, 0); break; default: DR_TMA(1, 1, 1); break;
        }
#undef DR_TMA
        CKL("k_pt_tma");
        H->cur ^= 1;
        if (H->form) H->stress_stale = true;
        return DR_OK;
    }
    const size_t smem = DrFusedCfg<FUSED_TX, FUSED_TY>::SMEM;
    DrConstFields A = cfields_of(H, H->cur);
    DrFields B = fields_of(H, H->cur ^ 1);
    if (H->gavg) { if (with_res) k_pt_fused<1, 1, FUSED_TX, FUSED_TY><<<grd, blk, smem, H->st>>>(H->L, P, A, B, H->K, H->G, lz, H->res_bits);
                   else          k_pt_fused<1, 0, FUSED_TX, FUSED_TY><<<grd, blk, smem, H->st>>>(H->L, P, A, B, H->K, H->G, lz, H->res_bits); }
    else         { if (with_res) k_pt_fused<0, 1, FUSED_TX, FUSED_TY><<<grd, blk, smem, H->st>>>(H->L, P, A, B, H->K, H->G, lz, H->res_bits);
                   else          k_pt_fused<0, 0, FUSED_TX, FUSED_TY><<<grd, blk, smem, H->st>>>(H->L, P, A, B, H->K, H->G, lz, H->res_bits); }
    CKL("k_pt_fused");
    H->cur ^= 1;
    return DR_OK;
}

// DR_KERNEL 3: iterations `it` and `it + 1` (1-based) go into ONE sweep when both fit below `last_allowed` and `it` is not
// itself a residual-check iteration (the sweep reports the residual of its second iteration only)
static int sweep_len(const dr_handle* H, int it, int last_allowed, int ncheck) {
    return (H->kernel == 3 && coded(H) && it + 1 <= last_allowed && (ncheck <= 0 || it % ncheck != 0)) ? 2 : 1;
}
static dr_status sweep(dr_handle* H, const DrPT& P, int n, bool with_res) {
    return n == 2 ? iteration_coded(H, P, with_res, 2) : iteration(H, P, with_res);
}

// buffer whose stress slots hold the stresses: in the displacement form the sigma_aa slots of the state buffer carry
// w, and the stresses (Hooke's law of the displacement BEFORE the last update, like the oracle's) sit in the other one
static int stress_buf(const dr_handle* H) { return H->form ? H->cur ^ 1 : H->cur; }

static dr_status ensure_stresses(dr_handle* H) {
    if (!H->form || !H->stress_stale) return DR_OK;
    const DrLayout& L = H->L;
    const DrPT P = make_pt(H, H->cur_lc, H->cur_eps0);
    const int b = H->cur ^ 1;                       // holds u before the last update; its w is dead
    dim3 blk(64, 4, 1), grd((L.nx + 1 + 63) / 64, (L.ny + 1 + 3) / 4, L.nz + 1);
    if (H->gavg) k_stress_split<1, 1><<<grd, blk, 0, H->st>>>(H->L, P, cfields_of(H, b), fields_of(H, b), H->K, H->G);
    else         k_stress_split<0, 1><<<grd, blk, 0, H->st>>>(H->L, P, cfields_of(H, b), fields_of(H, b), H->K, H->G);
    CKL("k_stress_split(finalize)");
    H->stress_stale = false;
    return DR_OK;
}

static dr_status read_residual(dr_handle* H, double* r) {
    CK(cudaMemcpyAsync(H->pinned + 8, H->res_bits, 8, cudaMemcpyDeviceToHost, H->st));
    CK(cudaStreamSynchronize(H->st));
    std::memcpy(r, H->pinned + 8, 8);
    return DR_OK;
}

// enqueue the volume averages (Eq. 7) and their copy into pinned[dst .. dst+5]; no synchronisation
static dr_status enqueue_averages(dr_handle* H, int dst) {
    const DrLayout& L = H->L;
    { dr_status es = ensure_stresses(H); if (es != DR_OK) return es; }
    k_avg_partial<<<DR_AVG_BLOCKS, DR_AVG_THREADS, 0, H->st>>>(H->L, cfields_of(H, stress_buf(H)), H->partial);
    CKL("k_avg_partial");
    k_avg_final<<<1, 256, 0, H->st>>>(H->partial, DR_AVG_BLOCKS, 1.0 / ((double)L.nx * L.ny * L.nz), H->avg_dev);
    CKL("k_avg_final");
    CK(cudaMemcpyAsync(H->pinned + dst, H->avg_dev, 6 * sizeof(double), cudaMemcpyDeviceToHost, H->st));
    return DR_OK;
}

static dr_status averages(dr_handle* H, int lc, double eps0) {
    { dr_status es = enqueue_averages(H, 0); if (es != DR_OK) return es; }
    CK(cudaEventRecord(H->e1, H->st));
    CK(cudaStreamSynchronize(H->st));
    for (int m = 0; m < 6; ++m) { H->avg[m] = H->pinned[m]; H->Ccol[lc][m] = H->avg[m] / eps0; }   // Eq. 9, 22
    H->have_avg = true; H->have[lc] = true;
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, H->e0, H->e1));
    H->ms = ms;
    return DR_OK;
}

// second stopping rule (Reading R9b): state of the <sigma> stagnation test of one solve
// The movement is taken over at least DR_STAG_WINDOW iterations, whatever DR_NCHECK is: a check closer than that to the
// last comparison is not `due` (with ncheck = 1 the per-iteration movement falls below stag_tol long before <sigma> has
// converged).  For ncheck >= 50 every check compares.
#define DR_STAG_WINDOW 50
struct DrStag {
    bool have_prev = false;
    double prev[6] = {0, 0, 0, 0, 0, 0};
    int calm = 0;
    int prev_it = 0;
    // does the check at iteration `it` take part in the rule (are its averages needed)?
    bool due(int it) const { return !have_prev || it - prev_it >= DR_STAG_WINDOW; }
    // a[6] = <sigma> at the check of iteration it (which is due); true when two consecutive comparisons moved <sigma> by
    // <= stag_tol (relative, max-norm)
    bool update(const double* a, double stag_tol, int it) {
        prev_it = it;
        double num = 0.0, den = 0.0;
        for (int m = 0; m < 6; ++m) { num = std::max(num, std::fabs(a[m] - prev[m])); den = std::max(den, std::fabs(a[m])); }
        if (have_prev && num <= stag_tol * den) ++calm; else calm = 0;
        for (int m = 0; m < 6; ++m) prev[m] = a[m];
        have_prev = true;
        return calm >= 2;
    }
};

static bool bad_lc(dr_handle* H, int lc, double eps0) {
    if (lc < 0 || lc > 6 || !(eps0 != 0.0) || !std::isfinite(eps0)) { H->err = "bad load case or eps0"; return true; }
    return false;
}

extern "C" dr_status dr_solve(dr_handle* H, int lc, double eps0, double tol, int maxiter) {
    if (!H) return DR_ERR_ARG;
    DrDeviceGuard dg(H->device);
    if (bad_lc(H, lc, eps0)) return DR_ERR_ARG;
    if (!(tol > 0.0) || maxiter < 1) return fail(H, DR_ERR_ARG, "bad tol or maxiter");
    CK(cudaEventRecord(H->e0, H->st));
    dr_status s = prepare(H, lc, eps0);
    if (s != DR_OK) return s;
    const DrPT P = make_pt(H, lc, eps0);
    dr_status status = DR_MAXITER;
    H->residual = INFINITY;
    H->stop_reason = DR_STOP_MAXITER;
    DrStag stag;
    const bool use_stag = H->stag_tol > 0.0;
    int it;
    for (it = 1; it <= maxiter; ++it) {
        const int n = sweep_len(H, it, maxiter, H->ncheck);
        it += n - 1;                                          // index of the last iteration of this sweep
        const bool chk = (it % H->ncheck == 0);
        if (chk) CK(cudaMemsetAsync(H->res_bits, 0, 8, H->st));
        s = sweep(H, P, n, chk);
        if (s != DR_OK) return s;
        if (chk) {
            // the averages of the stagnation rule ride on the same synchronisation as the residual
            const bool sdue = use_stag && stag.due(it);
            if (sdue) { s = enqueue_averages(H, 9); if (s != DR_OK) return s; }
            double r;
            s = read_residual(H, &r);
            if (s != DR_OK) return s;
            H->residual = r;
            if (!std::isfinite(r)) { status = DR_ERR_DIVERGED; H->stop_reason = DR_STOP_NONE; break; }
            if (r <= tol) { status = DR_OK; H->stop_reason = DR_STOP_RESIDUAL; break; }
            if (sdue && stag.update(H->pinned + 9, H->stag_tol, it)) { status = DR_OK; H->stop_reason = DR_STOP_STAGNATION; break; }
        }
    }
    H->iters = std::min(it, maxiter);
    if (status == DR_ERR_DIVERGED) {
        CK(cudaEventRecord(H->e1, H->st));
        CK(cudaStreamSynchronize(H->st));
        return fail(H, status, "residual is not finite");
    }
    s = averages(H, lc, eps0);
    if (s != DR_OK) return s;
    if (status == DR_MAXITER) H->err = "maxiter reached";
    return status;
}

// SURVEY 8(a) row a7 / north_star (c): the six load cases as six solvers on six streams.  One host thread enqueues, for
// every unfinished load case, the iterations up to its next residual check (no synchronisation), and only then waits
// for the six 8-byte residuals; small grids, whose single solve cannot fill the GPU, overlap on the device.
extern "C" dr_status dr_solve_six(dr_handle* const h[6], double eps0, double tol, int maxiter, int status_out[6]) {
    if (!h) return DR_ERR_ARG;
    for (int lc = 0; lc < 6; ++lc) {
        if (!h[lc]) return DR_ERR_ARG;
        for (int m = 0; m < lc; ++m) if (h[m] == h[lc]) return fail(h[lc], DR_ERR_ARG, "dr_solve_six needs six distinct handles");
        if (bad_lc(h[lc], lc, eps0)) return DR_ERR_ARG;
        if (!(tol > 0.0) || maxiter < 1) return fail(h[lc], DR_ERR_ARG, "bad tol or maxiter");
    }
    DrPT P[6];
    int it[6];
    bool active[6], pending[6], sdue[6] = {false, false, false, false, false, false};
    dr_status st[6];
    DrStag stag[6];
    for (int lc = 0; lc < 6; ++lc) {
        dr_handle* H = h[lc];
        DrDeviceGuard dg(H->device);
        H->stop_reason = DR_STOP_MAXITER;
        CK(cudaEventRecord(H->e0, H->st));
        dr_status s = prepare(H, lc, eps0);
        if (s != DR_OK) return s;
        P[lc] = make_pt(H, lc, eps0);
        it[lc] = 0; active[lc] = true; pending[lc] = false; st[lc] = DR_MAXITER; H->residual = INFINITY;
    }
    for (bool any = true; any;) {
        for (int lc = 0; lc < 6; ++lc) {
            if (!active[lc]) continue;
            dr_handle* H = h[lc];
            DrDeviceGuard dg(H->device);
            const int upto = it[lc] + std::min(H->ncheck - it[lc] % H->ncheck, maxiter - it[lc]);   // next check, or maxiter
            bool chk = false;
            while (it[lc] < upto) {
                const int n = sweep_len(H, it[lc] + 1, upto, H->ncheck);
                it[lc] += n;
                chk = (it[lc] % H->ncheck == 0);
                if (chk) CK(cudaMemsetAsync(H->res_bits, 0, 8, H->st));
                dr_status s = sweep(H, P[lc], n, chk);
                if (s != DR_OK) return s;
            }
            if (chk) {
                sdue[lc] = H->stag_tol > 0.0 && stag[lc].due(it[lc]);
                if (sdue[lc]) { dr_status s = enqueue_averages(H, 9); if (s != DR_OK) return s; }
                CK(cudaMemcpyAsync(H->pinned + 8, H->res_bits, 8, cudaMemcpyDeviceToHost, H->st));
            }
            pending[lc] = chk;
        }
        any = false;
        for (int lc = 0; lc < 6; ++lc) {
            if (!active[lc]) continue;
            dr_handle* H = h[lc];
            DrDeviceGuard dg(H->device);
            if (pending[lc]) {
                CK(cudaStreamSynchronize(H->st));
                double r;
                std::memcpy(&r, H->pinned + 8, 8);
                H->residual = r;
                if (!std::isfinite(r)) { st[lc] = DR_ERR_DIVERGED; active[lc] = false; H->stop_reason = DR_STOP_NONE; H->err = "residual is not finite"; }
                else if (r <= tol) { st[lc] = DR_OK; active[lc] = false; H->stop_reason = DR_STOP_RESIDUAL; }
                else if (sdue[lc] && stag[lc].update(H->pinned + 9, H->stag_tol, it[lc])) { st[lc] = DR_OK; active[lc] = false; H->stop_reason = DR_STOP_STAGNATION; }
            }
            if (active[lc] && it[lc] >= maxiter) { active[lc] = false; H->err = "maxiter reached"; }
            any = any || active[lc];
        }
    }
    dr_status worst = DR_OK;
    for (int lc = 0; lc < 6; ++lc) {
        dr_handle* H = h[lc];
        DrDeviceGuard dg(H->device);
        H->iters = it[lc];
        if (st[lc] != DR_ERR_DIVERGED) { dr_status s = averages(H, lc, eps0); if (s != DR_OK) return s; }
        if (status_out) status_out[lc] = (int)st[lc];
        if (st[lc] == DR_ERR_DIVERGED) worst = DR_ERR_DIVERGED;
        else if (st[lc] == DR_MAXITER && worst == DR_OK) worst = DR_MAXITER;
    }
    return worst;
}

// effective stiffness from six handles, column lc taken from h[lc] (after dr_solve_six)
extern "C" dr_status dr_effective_C_six(dr_handle* const h[6], double out[36]) {
    if (!h || !out) return DR_ERR_ARG;
    for (int lc = 0; lc < 6; ++lc) {
        if (!h[lc]) return DR_ERR_ARG;
        if (!h[lc]->have[lc]) return fail(h[lc], DR_ERR_STATE, "load case not solved on its handle");
    }
    for (int m = 0; m < 6; ++m) for (int lc = 0; lc < 6; ++lc) out[6 * m + lc] = h[lc]->Ccol[lc][m];
    return DR_OK;
}

// the six load cases of one image advanced TOGETHER -- every launch of the two-iteration kernel
// carries all unfinished load cases (they share the stencil codes; one direct test per stiffness column).
// Same iterates, residual checks, stagnation rule and C as six dr_solve calls.
extern "C" dr_status dr_solve_all(dr_handle* H, double eps0, double tol, int maxiter, int status_out[6]) {
    if (!H) return DR_ERR_ARG;
    DrDeviceGuard dg(H->device);
    if (bad_lc(H, 0, eps0)) return DR_ERR_ARG;
    if (!(tol > 0.0) || maxiter < 1) return fail(H, DR_ERR_ARG, "bad tol or maxiter");
    if (H->nsets != 6) return fail(H, DR_ERR_WORKSPACE, "dr_solve_all needs a workspace of dr_workspace_bytes_six() bytes at dr_create");
    CK(cudaEventRecord(H->e0, H->st));
    { dr_status ms = prepare_moduli(H); if (ms != DR_OK) return ms; }
    dr_status worst = DR_OK;
    if (!(H->kernel == 3 && coded(H))) {
        // not a stencil-coded image (or another kernel / form chosen): the six solves one after the other on state set 0
        for (int lc = 0; lc < 6; ++lc) {
            dr_status s = dr_solve(H, lc, eps0, tol, maxiter);
            H->lc_iters[lc] = H->iters; H->lc_res[lc] = H->residual; H->lc_stop[lc] = H->stop_reason;
            if (status_out) status_out[lc] = (int)s;
            if (s != DR_OK && s != DR_MAXITER) {
                // hard error: the load cases that never ran report DR_ERR_STATE / no iterations instead of stale values
                for (int m = lc + 1; m < 6; ++m) {
                    H->lc_iters[m] = 0; H->lc_res[m] = INFINITY; H->lc_stop[m] = DR_STOP_NONE;
                    if (status_out) status_out[m] = (int)DR_ERR_STATE;
                }
                return s;
            }
            if (s == DR_MAXITER) worst = DR_MAXITER;
        }
        return worst;
    }
    const DrLayout& L = H->L;
    DrPT P[6];
    int cur[6];
    bool active[6];
    dr_status st[6];
    DrStag stag[6];
    for (int lc = 0; lc < 6; ++lc) {
        P[lc] = make_pt(H, lc, eps0);
        DrFields F; for (int f = 0; f < F_COUNT; ++f) F.f[f] = H->xbuf[lc][0][f];
        dim3 blk(32, 4, 1), grd(((L.nx + 3) / 2 + 31) / 32, (L.ny + 1 + 3) / 4, (L.nz + 1 + DR_BC_ZB - 1) / DR_BC_ZB);   // pairs (2t-1, 2t), t = 0 .. (nx+2)/2
        if (H->gavg) k_bc_init<1><<<grd, blk, 0, H->st>>>(H->L, P[lc], F, F, 0, H->K, H->G);
        else         k_bc_init<0><<<grd, blk, 0, H->st>>>(H->L, P[lc], F, F, 0, H->K, H->G);
        CKL("k_bc_init");
        cur[lc] = 0; active[lc] = true; st[lc] = DR_MAXITER;
        H->lc_iters[lc] = 0; H->lc_res[lc] = INFINITY; H->lc_stop[lc] = DR_STOP_MAXITER; H->have[lc] = false;
    }
    H->have_fields = false;                          // set 0 now holds load case 0 of the batch, not a dr_step state
    static thread_local DrTb2Batch TB;
    const bool use_stag = H->stag_tol > 0.0;
    const double invN = 1.0 / ((double)L.nx * L.ny * L.nz);
    int it = 0, nact = 6;
    while (nact > 0 && it < maxiter) {
        const int n = (it + 2 <= maxiter && (it + 1) % H->ncheck != 0) ? 2 : 1;
        it += n;
        const bool chk = (it % H->ncheck == 0);
        int slots[6], ns = 0;
        for (int lc = 0; lc < 6; ++lc) if (active[lc]) { fill_slot(H, TB, ns, lc, cur[lc], P[lc]); slots[ns++] = lc; }
        if (chk) CK(cudaMemsetAsync(H->res_bits, 0, 6 * 8, H->st));
        { dr_status s = launch_coded(H, TB, ns, chk, n); if (s != DR_OK) return s; }
        for (int a = 0; a < ns; ++a) cur[slots[a]] ^= 1;
        if (!chk) continue;
        const bool sdue = use_stag && stag[slots[0]].due(it);     // the active load cases share their comparison history
        if (sdue) {
            DrAvgSix A;
            for (int a = 0; a < ns; ++a) for (int f = 0; f < F_COUNT; ++f) A.F[a].f[f] = H->xbuf[slots[a]][cur[slots[a]]][f];
            k_avg_partial6<<<dim3(DR_AVG_BLOCKS, ns), DR_AVG_THREADS, 0, H->st>>>(H->L, A, H->partial6);
            CKL("k_avg_partial6");
            k_avg_final6<<<ns, 256, 0, H->st>>>(H->partial6, DR_AVG_BLOCKS, invN, H->avg6_dev);
            CKL("k_avg_final6");
            CK(cudaMemcpyAsync(H->pinned + 24, H->avg6_dev, (size_t)ns * 6 * sizeof(double), cudaMemcpyDeviceToHost, H->st));
        }
        CK(cudaMemcpyAsync(H->pinned + 16, H->res_bits, 6 * 8, cudaMemcpyDeviceToHost, H->st));
        CK(cudaStreamSynchronize(H->st));
        for (int a = 0; a < ns; ++a) {
            const int lc = slots[a];
            double r;
            std::memcpy(&r, H->pinned + 16 + lc, 8);
            H->lc_res[lc] = r;
            bool done = false;
            if (!std::isfinite(r)) { st[lc] = DR_ERR_DIVERGED; H->lc_stop[lc] = DR_STOP_NONE; done = true; }
            else if (r <= tol) { st[lc] = DR_OK; H->lc_stop[lc] = DR_STOP_RESIDUAL; done = true; }
            else if (sdue && stag[lc].update(H->pinned + 24 + 6 * a, H->stag_tol, it)) { st[lc] = DR_OK; H->lc_stop[lc] = DR_STOP_STAGNATION; done = true; }
            if (done) { active[lc] = false; H->lc_iters[lc] = it; --nact; }
        }
    }
    for (int lc = 0; lc < 6; ++lc) if (active[lc]) H->lc_iters[lc] = it;
    // volume averages of all six final states (Eq. 7) -> the six columns (Eq. 9, 22)
    {
        DrAvgSix A;
        for (int lc = 0; lc < 6; ++lc) for (int f = 0; f < F_COUNT; ++f) A.F[lc].f[f] = H->xbuf[lc][cur[lc]][f];
        k_avg_partial6<<<dim3(DR_AVG_BLOCKS, 6), DR_AVG_THREADS, 0, H->st>>>(H->L, A, H->partial6);
        CKL("k_avg_partial6");
        k_avg_final6<<<6, 256, 0, H->st>>>(H->partial6, DR_AVG_BLOCKS, invN, H->avg6_dev);
        CKL("k_avg_final6");
        CK(cudaMemcpyAsync(H->pinned + 24, H->avg6_dev, 36 * sizeof(double), cudaMemcpyDeviceToHost, H->st));
        CK(cudaEventRecord(H->e1, H->st));
        CK(cudaStreamSynchronize(H->st));
    }
    for (int lc = 0; lc < 6; ++lc) {
        if (status_out) status_out[lc] = (int)st[lc];
        if (st[lc] == DR_ERR_DIVERGED) { worst = DR_ERR_DIVERGED; continue; }
        for (int m = 0; m < 6; ++m) H->Ccol[lc][m] = H->pinned[24 + 6 * lc + m] / eps0;
        H->have[lc] = true;
        if (st[lc] == DR_MAXITER && worst == DR_OK) worst = DR_MAXITER;
    }
    for (int m = 0; m < 6; ++m) H->avg[m] = H->pinned[24 + 30 + m];
    H->have_avg = true;
    H->iters = H->lc_iters[5]; H->residual = H->lc_res[5]; H->stop_reason = H->lc_stop[5];
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, H->e0, H->e1));
    H->ms = ms;
    if (worst == DR_MAXITER) H->err = "maxiter reached";
    if (worst == DR_ERR_DIVERGED) H->err = "residual is not finite";
    return worst;
}

// iterations, last residual and dr_stop of load case lc in the last dr_solve_all
extern "C" dr_status dr_info_lc(dr_handle* H, int lc, int* iters, double* residual, int* stop) {
    if (!H || lc < 0 || lc > 5) return DR_ERR_ARG;
    if (iters) *iters = H->lc_iters[lc];
    if (residual) *residual = H->lc_res[lc];
    if (stop) *stop = H->lc_stop[lc];
    return DR_OK;
}

extern "C" dr_status dr_step(dr_handle* H, int lc, double eps0, int niter) {
    if (!H) return DR_ERR_ARG;
    DrDeviceGuard dg(H->device);
    if (bad_lc(H, lc, eps0)) return DR_ERR_ARG;
    if (niter < 0) return fail(H, DR_ERR_ARG, "bad niter");
    CK(cudaEventRecord(H->e0, H->st));
    dr_status s = prepare(H, lc, eps0);
    if (s != DR_OK) return s;
    const DrPT P = make_pt(H, lc, eps0);
    double r = 0.0;
    for (int it = 1; it <= niter; ++it) {
        const int n = sweep_len(H, it, niter, 0);
        it += n - 1;
        const bool last = (it == niter);
        if (last) CK(cudaMemsetAsync(H->res_bits, 0, 8, H->st));
        s = sweep(H, P, n, last);
        if (s != DR_OK) return s;
    }
    if (niter > 0) { s = read_residual(H, &r); if (s != DR_OK) return s; }
    H->iters = niter; H->residual = r;
    return averages(H, lc, eps0);
}

extern "C" dr_status dr_iterate(dr_handle* H, int lc, double eps0, int niter) {
    if (!H) return DR_ERR_ARG;
    DrDeviceGuard dg(H->device);
    if (bad_lc(H, lc, eps0)) return DR_ERR_ARG;
    if (niter < 0) return fail(H, DR_ERR_ARG, "bad niter");
    if (!H->have_fields || lc != H->cur_lc || eps0 != H->cur_eps0)
        return fail(H, DR_ERR_STATE, "dr_iterate needs a previous dr_step/dr_solve with the same load case and eps0");
    const DrPT P = make_pt(H, lc, eps0);
    for (int it = 1; it <= niter; ++it) {
        const int n = sweep_len(H, it, niter, 0);
        it += n - 1;
        dr_status s = sweep(H, P, n, false);
        if (s != DR_OK) return s;
    }
    return DR_OK;
}

extern "C" dr_status dr_effective_C(dr_handle* H, double out[36]) {
    if (!H || !out) return DR_ERR_ARG;
    for (int lc = 0; lc < 6; ++lc) if (!H->have[lc]) return fail(H, DR_ERR_STATE, "not all six load cases solved");
    for (int m = 0; m < 6; ++m) for (int lc = 0; lc < 6; ++lc) out[6 * m + lc] = H->Ccol[lc][m];
    return DR_OK;
}

// Eq. 24-29: C12, C13, C23 from the 7th (triaxial) direct test, load case 6, and C11, C22, C33 of the normal
// tests.  Ccol holds <sigma>/eps0, so with eps_bar_k = eps0 (Eq. 25) the strains cancel: sigma_bar_k / eps0 = Ccol[6][k] - C_kk.
extern "C" dr_status dr_offdiag_direct(dr_handle* H, double out[3]) {
    if (!H || !out) return DR_ERR_ARG;
    static const int need[4] = {0, 1, 2, 6};
    for (int q = 0; q < 4; ++q) if (!H->have[need[q]]) return fail(H, DR_ERR_STATE, "dr_offdiag_direct needs load cases 0, 1, 2 and 6");
    const double sb1 = H->Ccol[6][0] - H->Ccol[0][0], sb2 = H->Ccol[6][1] - H->Ccol[1][1], sb3 = H->Ccol[6][2] - H->Ccol[2][2];
    out[0] = 0.5 * (sb1 + sb2 - sb3);      // Eq. 27
    out[1] = 0.5 * (sb1 - sb2 + sb3);      // Eq. 28
    out[2] = 0.5 * (-sb1 + sb2 + sb3);     // Eq. 29
    return DR_OK;
}

extern "C" dr_status dr_avg_stress(dr_handle* H, double out[6]) {
    if (!H || !out) return DR_ERR_ARG;
    if (!H->have_avg) return fail(H, DR_ERR_STATE, "no solve yet");
    for (int m = 0; m < 6; ++m) out[m] = H->avg[m];
    return DR_OK;
}

extern "C" dr_status dr_info(dr_handle* H, int* iters, double* residual, double* ms) {
    if (!H) return DR_ERR_ARG;
    if (iters) *iters = H->iters;
    if (residual) *residual = H->residual;
    if (ms) *ms = H->ms;
    return DR_OK;
}

extern "C" dr_status dr_get_field(dr_handle* H, int field, double* dst, size_t n) {
    if (!H || !dst) return DR_ERR_ARG;
    DrDeviceGuard dg(H->device);
    if (field < 0 || field >= F_COUNT) return fail(H, DR_ERR_ARG, "bad field id");
    if (!H->have_fields) return fail(H, DR_ERR_STATE, "no fields yet");
    const DrLayout& L = H->L;
    int ex = L.nx, ey = L.ny, ez = L.nz;
    switch (field) {
        case F_VX: ex++; break; case F_VY: ey++; break; case F_VZ: ez++; break;
        case F_TYZ: ey++; ez++; break; case F_TXZ: ex++; ez++; break; case F_TXY: ex++; ey++; break;
        default: break;
    }
    if (n != (size_t)ex * ey * ez) return fail(H, DR_ERR_ARG, "bad field size");
    dim3 blk(64, 4, 1), grd((ex + 63) / 64, (ey + 3) / 4, ez);
    { dr_status es = ensure_stresses(H); if (es != DR_OK) return es; }
    const int src = field <= F_VZ ? H->cur : stress_buf(H);
    k_export<<<grd, blk, 0, H->st>>>(H->L, H->buf[src][field], dst, ex, ey, ez);
    CKL("k_export");
    CK(cudaStreamSynchronize(H->st));
    return DR_OK;
}

// the six load cases of a freshly created handle -> C_out; destroys the handle
static dr_status solve_image(dr_handle* H, double eps0, double tol, int maxiter, int ncheck, double C_out[36], int iters_out[6]) {
    dr_status s, worst = DR_OK;
    if (ncheck > 0) dr_set_param(H, DR_NCHECK, ncheck);
    if (H->nsets == 6) {                             // workspace of dr_workspace_bytes_six: all six load cases per launch
        s = dr_solve_all(H, eps0, tol, maxiter, nullptr);
        if (iters_out) for (int lc = 0; lc < 6; ++lc) iters_out[lc] = H->lc_iters[lc];
        if (s != DR_OK && s != DR_MAXITER) { dr_destroy(H); return s; }
        worst = s;
    } else
    for (int lc = 0; lc < 6; ++lc) {
        s = dr_solve(H, lc, eps0, tol, maxiter);
        if (iters_out) iters_out[lc] = H->iters;
        if (s != DR_OK && s != DR_MAXITER) { dr_destroy(H); return s; }
        if (s == DR_MAXITER) worst = DR_MAXITER;
    }
    s = dr_effective_C(H, C_out);
    dr_destroy(H);
    return s != DR_OK ? s : worst;
}

extern "C" dr_status dr_solve_image_host(int nx, int ny, int nz, double h, const double* K_host, const double* G_host,
                                         double* stage_device, void* workspace, size_t workspace_bytes, void* cuda_stream,
                                         double eps0, double tol, int maxiter, int ncheck, double C_out[36], int iters_out[6]) {
    if (!sizes_ok(nx, ny, nz) || !K_host || !G_host || !stage_device || !C_out) return DR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t N = (size_t)nx * ny * nz;
    if (cudaMemcpyAsync(stage_device, K_host, N * sizeof(double), cudaMemcpyHostToDevice, st) != cudaSuccess) return DR_ERR_CUDA;
    if (cudaMemcpyAsync(stage_device + N, G_host, N * sizeof(double), cudaMemcpyHostToDevice, st) != cudaSuccess) return DR_ERR_CUDA;
    dr_handle* H = nullptr;
    dr_status s = dr_create(nx, ny, nz, h, stage_device, stage_device + N, workspace, workspace_bytes, cuda_stream, &H);
    if (s != DR_OK) return s;
    return solve_image(H, eps0, tol, maxiter, ncheck, C_out, iters_out);
}

extern "C" dr_status dr_solve_image_host_segmented(int nx, int ny, int nz, double h, const unsigned char* phase_host, int nphase,
                                                   const double* K_table, const double* G_table,
                                                   unsigned char* stage_device, void* workspace, size_t workspace_bytes, void* cuda_stream,
                                                   double eps0, double tol, int maxiter, int ncheck, double C_out[36], int iters_out[6]) {
    if (!sizes_ok(nx, ny, nz) || !phase_host || !stage_device || !C_out) return DR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t N = (size_t)nx * ny * nz;
    if (cudaMemcpyAsync(stage_device, phase_host, N, cudaMemcpyHostToDevice, st) != cudaSuccess) return DR_ERR_CUDA;
    dr_handle* H = nullptr;
    dr_status s = dr_create_segmented(nx, ny, nz, h, stage_device, nphase, K_table, G_table, workspace, workspace_bytes, cuda_stream, &H);
    if (s != DR_OK) return s;
    return solve_image(H, eps0, tol, maxiter, ncheck, C_out, iters_out);
}

// 6x6 inverse by Gauss-Jordan elimination with partial pivoting (host); false if singular
static bool invert6(const double* A, double* inv) {
    double a[6][12];
    for (int r = 0; r < 6; ++r) for (int c = 0; c < 6; ++c) { a[r][c] = A[6 * r + c]; a[r][6 + c] = (r == c) ? 1.0 : 0.0; }
    for (int c = 0; c < 6; ++c) {
        int piv = c;
        for (int r = c + 1; r < 6; ++r) if (std::fabs(a[r][c]) > std::fabs(a[piv][c])) piv = r;
        if (!(std::fabs(a[piv][c]) > 0.0) || !std::isfinite(a[piv][c])) return false;
        if (piv != c) for (int k = 0; k < 12; ++k) std::swap(a[piv][k], a[c][k]);
        const double d = 1.0 / a[c][c];
        for (int k = 0; k < 12; ++k) a[c][k] *= d;
        for (int r = 0; r < 6; ++r) {
            if (r == c) continue;
            const double f = a[r][c];
            if (f != 0.0) for (int k = 0; k < 12; ++k) a[r][k] -= f * a[c][k];
        }
    }
    for (int r = 0; r < 6; ++r) for (int c = 0; c < 6; ++c) inv[6 * r + c] = a[r][6 + c];
    return true;
}

// Eq. 23: S* = S1 + phi H  =>  H = ((C*)^-1 - (C1)^-1) / phi, host post-processing of two results
extern "C" dr_status dr_contribution_tensor(const double C_eff[36], const double C_matrix[36], double phi, double H_out[36]) {
    if (!C_eff || !C_matrix || !H_out || !(phi > 0.0) || !(phi <= 1.0)) return DR_ERR_ARG;
    double Se[36], S1[36];
    if (!invert6(C_eff, Se) || !invert6(C_matrix, S1)) return DR_ERR_ARG;
    for (int a = 0; a < 36; ++a) H_out[a] = (Se[a] - S1[a]) / phi;
    return DR_OK;
}

extern "C" int dr_uses_palette(dr_handle* H) { return (H && H->has_pal && H->use_pal && (H->kernel == 0 || H->kernel >= 3)) ? 1 : 0; }

// kernel that the iterations of the last dr_step / dr_solve really ran: DR_KERNEL, except that 3 and 4 report 0 when the
// image could not be stencil-coded (more than 256 distinct cell pairs, edge moduli or node stiffnesses)
extern "C" int dr_active_kernel(dr_handle* H) { return !H ? -1 : (H->kernel >= 3 && !coded(H) ? 0 : H->kernel); }

extern "C" long long dr_launch_count(dr_handle* H) { return H ? H->launches : 0; }

extern "C" const char* dr_last_error(dr_handle* H) { return H ? H->err.c_str() : "null handle"; }

extern "C" int dr_stop_reason(dr_handle* H) { return H ? H->stop_reason : (int)DR_STOP_NONE; }

extern "C" void dr_destroy(dr_handle* H) {
    if (!H) return;
    DrDeviceGuard dg(H->device);
    cudaStreamSynchronize(H->st);
    pinned_release(H->pinned);
    if (H->e0) cudaEventDestroy(H->e0);
    if (H->e1) cudaEventDestroy(H->e1);
    delete H;
}
