// dr_kernels_tb2.cuh -- TWO PT iterations per sweep (temporal blocking, BASELINE north_star "optional
// temporal blocking") on "stencil-coded" images.
//
// Why: the one-sweep kernel k_pt_tma moves its 160 B per voxel-iteration at ~0.8 of the copy rate; the only way past the
// DRAM rate is to advance the state by two iterations while it is on chip ("performance ... depends on the GPU
// bandwidth").  One launch of k_pt_tb2<.,2,..> reads the state of iteration n once and writes that of iteration n+2 once.
//
// What makes it fit (registers, shared memory, issue slots): everything that depends on the moduli only is taken out of
// the iteration.  A segmented image has few distinct (K,G) pairs, hence few distinct edge shear moduli (means of 4 cells)
// and few distinct node stiffnesses H_node (max of six springs).  dr_code_* (below) tabulates, ONCE per (image, DR_GAVG,
// DR_VOID_REL): the distinct cell pairs (the palette of dr_kernels_aux.cuh), the distinct edge moduli E[256] and the
// distinct 1/H_node values R[256] (0 for wall / dead / out-of-domain nodes), and gives every node of every tile a 64-bit
// stencil code = 7 table indices:
//     byte 0  cell (K,G) of cell (i,j,k)          byte 4  1/H_node of the v_x node (i, j+1/2, k+1/2)
//     byte 1  G_xy of edge (i, j, k+1/2)           byte 5  1/H_node of the v_y node (i+1/2, j, k+1/2)
//     byte 2  G_xz of edge (i, j+1/2, k+1)         byte 6  1/H_node of the v_z node (i+1/2, j+1/2, k)
//     byte 3  G_yz of edge (i+1/2, j, k+1)
// The table values are produced by the very functions the one-sweep kernel evaluates on the fly (dr_edge_mean_fast,
// dr_rcp), so the iterates are the same numbers.  With them the iteration needs no harmonic means, no reciprocals, no
// neighbour moduli (4 of the 9 exchange planes and 5 of the 10 carried doubles of k_pt_tma disappear) and no wall tests.
// More than 256 distinct values of any kind: the image is not coded and DR_KERNEL 3 runs the one-sweep kernel.
//
// Geometry: a CTA of TX x TY threads owns the (TX-4) x (TY-4) inner tile of a TX x TY extended tile (halo 2) and a chunk
// of z layers; thread (tx,ty) owns one node column.  z-march as in k_pt_tma; per step k (two barriers):
//     phase alpha:  A2(k-2): new stresses of the SECOND iteration for layer k-2, from the first iteration's velocities of
//                            layers k-2, k-1 (shared planes V1) and its stresses of layer k-2 (still in X1 from step k-2)
//                   A1(k):   new stresses of the FIRST iteration for layer k, from the TMA rings (old state) -> X1
//     phase beta:   B2(k-2): second-iteration velocities of layer k-2 -> the 9 output fields of layer k-2 (global stores)
//                   B1(k):   first-iteration velocities of layer k -> V1 (never leave the SM)
// First-iteration results are valid on the extended tile minus one ring, second-iteration results on the inner tile.
// A chunk [kb, ke) runs steps k = kb-2 .. ke+1 (iteration 1 on layers kb-2 .. ke, iteration 2 on kb-1 .. ke-1).
#pragma once
#include "dr_kernels_tma.cuh"

#ifndef TB2_TX
#define TB2_TX 32
#endif
#ifndef TB2_TY
#define TB2_TY 16
#endif
#ifndef TB2_UNROLL4
#define TB2_UNROLL4 0      // 1: march unrolled by 4 (every ring slot a compile-time constant); 0: by 2 (ring-A slot at run time)
#endif
#ifndef TB2_REREAD
#define TB2_REREAD 0       // 1: B2 reads its own second-iteration stresses back from the exchange planes; 0: keeps them in registers
#endif
#ifndef TB2_SKIPA2
#define TB2_SKIPA2 1       // 1: the outermost rows of the extended tile skip the second-iteration stress update (nobody reads it)
#endif
#ifndef TB2_LG128
#define TB2_LG128 0        // 1: lambda and 2G of a cell come with one 16-byte table read
#endif
#ifndef TB2_CTAB
#define TB2_CTAB 1         // 1: the derived tables travel in the kernel parameters and are read with LDC (constant cache, indexed per
                           //    thread) instead of from shared memory: 16 table reads per thread and step leave the shared-memory pipe
#endif
#define TB2_KLO 2          // coded layers below layer 0 (layers -2, -1) ...
#define TB2_KHI 3          // ... and above layer nz-1 (layers nz, nz+1, nz+2)

// tables of one coded image (global memory): K[256] G[256] (cell palette, after the void clamp), E[256] edge moduli,
// R[256] 1/H_node
#define TB2_TAB_K 0
#define TB2_TAB_G 256
#define TB2_TAB_E 512
#define TB2_TAB_R 768
#define TB2_TAB_N 1024
// the derived tables (TB2_CTAB: formed on the host per launch and passed in the kernel parameters, read with per-thread
// indexed LDC; else built by every CTA in shared memory): the products that are the same in every iteration
//   LAM = K - 2G/3,  G2 = 2G (interleaved, entry e at 2e and 2e+1, when TB2_LG128),  ES = (theta/h) E,  CV = (C~^2 h^2 / (theta h)) R,  RH = R (residual launches only)
#define TB2_S_LAM 0
#define TB2_S_G2 256
#define TB2_S_ES 512
#define TB2_S_CV 768
#define TB2_S_RH 1024

// One launch advances up to six load cases of the same image ("slots"; they share the stencil codes and tables, P:142-149:
// one direct test per stiffness column): blockIdx.z = slot * nchunks + z chunk.  A single solve is a batch of one.
#define TB2_NLC 6
struct DrTb2Batch {
    CUtensorMap m[TB2_NLC][9];            // per slot: vx vy vz | sxx syy szz txy | txz tyz of the OLD state (boxes TX x TY x 1)
    double* out[TB2_NLC];                 // per slot: field 0 (vx) of the NEW state; the other fields follow at stride fs
    unsigned long long* res[TB2_NLC];     // per slot: residual max-norm (bit pattern, atomicMax)
    DrPT P[TB2_NLC];                      // per slot: constants of its load case
    long long fs;                         // doubles between consecutive fields of a state buffer
    const unsigned long long* codes;      // [nz + KLO + KHI][gy][gx][TY][TX] stencil codes, layer -KLO first
    const double* tabs;                   // TB2_TAB_N doubles
    int gx, gy, nchunks;
    unsigned long long l2_hint;
#if TB2_CTAB
    double dtab[1280];                    // derived tables TB2_S_* (LAM G2 ES CV RH), formed on the host from tabs
#endif
};
// what the march needs of one slot
struct DrTb2Maps {
    const CUtensorMap* m;
    unsigned long long l2_hint;
};

// shared-memory exchange planes: X1 first-iteration stresses (double-buffered by step parity: the buffer written at step k
// still holds layer k-2 when step k starts, which is exactly what A2(k-2) needs), X2 second-iteration stresses
enum { Y_SXX = 0, Y_SYY, Y_TXY, Y_TXZ, Y_TYZ, Y_SZZ, Y_COUNT };
enum { Z_SXX = 0, Z_SYY, Z_TXY, Z_TXZ, Z_TYZ, Z_COUNT };

template <int TX, int TY>
struct DrTb2Cfg {
    static constexpr int PL = TX * TY;                       // doubles per plane
    static constexpr int NA = 4;                             // ring A slot: vx vy vz + stencil codes
    static constexpr int NB = 6;                             // ring B slot: sxx syy szz txy (layer m-1), txz tyz (face m)
    static constexpr int FRONT = 128;
    static constexpr int RING_A = FRONT;                     // [4][NA][PL]
    static constexpr int RING_B = RING_A + 4 * NA * PL;      // [2][NB][PL]
    static constexpr int X1 = RING_B + 2 * NB * PL;          // [2][Y_COUNT][PL]
    static constexpr int V1 = X1 + 2 * Y_COUNT * PL;         // [2][3][PL]
    static constexpr int X2 = V1 + 2 * 3 * PL;               // [Z_COUNT][PL]
    static constexpr int END = X2 + Z_COUNT * PL;
    static constexpr size_t SMEM = (size_t)(END + 64) * sizeof(double);
    static constexpr unsigned BYTES_A = NA * PL * sizeof(double);
    static constexpr unsigned BYTES_B = NB * PL * sizeof(double);
};

struct DrStress6 { double sxx, syy, szz, txy, txz, tyz; };
struct DrFace5 { double txz, tyz, szz, txz_r, tyz_u; };        // face values carried from one step to the next

// Stage A of one PT iteration at node column (i,j), layer k (Eq. 12-13, relaxation term implicit): new normal
// stresses and tau_xy of layer k, tau_xz / tau_yz of face k+1, from the velocities of layers k ("c") and k+1 ("n").
// Same expressions as stage A of dr_tma_step (FORM 0), except that the 1/h of the strain rates is folded into the
// constants (thh = theta/h, es = theta/h x edge modulus): identical bits for h = 1, last-bit differences otherwise.
template <bool BND>
__device__ __forceinline__ DrStress6 dr_tb2_stress(const DrPT& P, const int nx, const int ny, const int nz,
                                                   const int i, const int j, const int k,
                                                   const double lam, const double g2, const double esxy, const double esxz, const double esyz,
                                                   const double vxc, const double vyc, const double vzc,
                                                   const double vx_r, const double vy_u, const double vx_d, const double vy_l,
                                                   const double vxn, const double vyn, const double vzn,
                                                   const double vzn_l, const double vzn_d, const DrStress6& o) {
    const double h = P.h, ri = P.rinv, thh = P.theta * P.inv_h;
    DrStress6 n;
    const double dxx = vx_r - vxc;
    const double dyy = vy_u - vyc;
    const double dzz = vzn - vzc;
    const double lam_div = lam * (dxx + dyy + dzz);
    n.sxx = (o.sxx + thh * fma(g2, dxx, lam_div)) * ri;
    n.syy = (o.syy + thh * fma(g2, dyy, lam_div)) * ri;
    n.szz = (o.szz + thh * fma(g2, dzz, lam_div)) * ri;
    double exy = (vxc - vx_d) + (vyc - vy_l);
    double exz = (vxn - vxc) + (vzn - vzn_l);
    double eyz = (vyn - vyc) + (vzn - vzn_d);
    const bool bk1 = (k + 1 == 0 || k + 1 == nz);
    bool zxy = false, zxz = bk1, zyz = bk1;
    if (BND) {
        const bool bi = (i == 0 || i == nx), bj = (j == 0 || j == ny);
        zxy = bi | bj; zxz |= bi; zyz |= bj;
    }
    // boundary edges: stress free, or ghost rule when that component is prescribed on the faces
    if (zxy && P.ghost_xy) {
        const double z = (k + 0.5) * h;
        exy = dr_dshear(vxc, vx_d, j, ny, dr_u0(P, 0, i * h, j == 0 ? 0.0 : P.Ly, z))
            + dr_dshear(vyc, vy_l, i, nx, dr_u0(P, 1, i == 0 ? 0.0 : P.Lx, j * h, z));
        zxy = false;
    }
    if (zxz && P.ghost_xz) {
        const double y = (j + 0.5) * h;
        exz = dr_dshear(vxn, vxc, k + 1, nz, dr_u0(P, 0, i * h, y, k + 1 == 0 ? 0.0 : P.Lz))
            + dr_dshear(vzn, vzn_l, i, nx, dr_u0(P, 2, i == 0 ? 0.0 : P.Lx, y, (k + 1) * h));
        zxz = false;
    }
    if (zyz && P.ghost_yz) {
        const double x = (i + 0.5) * h;
        eyz = dr_dshear(vyn, vyc, k + 1, nz, dr_u0(P, 1, x, j * h, k + 1 == 0 ? 0.0 : P.Lz))
            + dr_dshear(vzn, vzn_d, j, ny, dr_u0(P, 2, x, j == 0 ? 0.0 : P.Ly, (k + 1) * h));
        zyz = false;
    }
    n.txy = zxy ? 0.0 : fma(esxy, exy, o.txy) * ri;
    n.txz = zxz ? 0.0 : fma(esxz, exz, o.txz) * ri;
    n.tyz = zyz ? 0.0 : fma(esyz, eyz, o.tyz) * ri;
    return n;
}

// entry of derived table SEC (TB2_S_*) at byte offset off8 = 8 x index
#if TB2_CTAB
#define TB2_TAB(SEC, off8) (*reinterpret_cast<const double*>(reinterpret_cast<const char*>(TB.dtab + (SEC)) + (off8)))
#else
#define TB2_TAB(SEC, off8) (*reinterpret_cast<const double*>(reinterpret_cast<const char*>(tab + (SEC)) + (off8)))
#endif

// velocity update of one node (Eq. 11): v += C~^2 h^2 / (theta H_node) F, with F = Fh / h the stress divergence;
// cv = C~^2 h^2 / (theta h H_node) and rH = 1/H_node from the tables, both 0 for wall, dead and out-of-domain nodes
// (never updated, not part of the residual).  rmax collects |Fh| / H_node (scaled by 1/h and h/|eps0| at the end).
template <int RES>
__device__ __forceinline__ double dr_tb2_vel(const double v, const double Fh, const DrTb2Batch& TB, const double* tab, const unsigned idx8, double& rmax, bool& rnan) {
    const double cv = TB2_TAB(TB2_S_CV, idx8);
    if (RES) {
        const double r = fabs(Fh) * TB2_TAB(TB2_S_RH, idx8);
        if (cv != 0.0) { rnan |= !(r == r); rmax = dr_max(rmax, r); }
    }
    return cv != 0.0 ? fma(cv, Fh, v) : v;
}

// byte b of a stencil code as a byte offset into a table of doubles
__device__ __forceinline__ unsigned dr_code_off(const unsigned long long c, const int b) {
    return b == 0 ? ((unsigned)c << 3) & 0x7f8u : (unsigned)(c >> (8 * b - 3)) & 0x7f8u;
}
__device__ __forceinline__ double dr_tab_at(const double* tab, const unsigned off8) {
    return *reinterpret_cast<const double*>(reinterpret_cast<const char*>(tab) + off8);
}

// lambda = K - 2G/3 and 2G of the cell whose table offset (index x 8) is off8
__device__ __forceinline__ void dr_tab_lg(const DrTb2Batch& TB, const double* tab, const unsigned off8, double& lam, double& g2) {
#if TB2_LG128 && !TB2_CTAB
    const double2 v = *reinterpret_cast<const double2*>(reinterpret_cast<const char*>(tab) + 2u * off8);    // interleaved: one 16-byte read
    lam = v.x; g2 = v.y;
#else
    lam = TB2_TAB(TB2_S_LAM, off8); g2 = TB2_TAB(TB2_S_G2, off8);
#endif
}

// TMA group u (u >= 0): what step u needs and no earlier step has brought: ring-A planes of layer m = k_u + 1 (velocities +
// codes; slot (u+1) & 3) and the old stresses of step u (sxx syy szz txy of layer m-1, txz tyz of face m; ring-B slot u & 1).
// Group -1 is ring-A layer kb-2 alone.  Completion: mbarrier (u+1) & 3, phase ((u+1) >> 2) & 1.
template <int TX, int TY>
__device__ __forceinline__ void dr_tb2_issue_group(const DrTb2Maps& T, unsigned long long* bars, double* sm,
                                                   const unsigned long long* codesrc, long long codestride,
                                                   int x0, int y0, int u, int m) {
    using Cfg = DrTb2Cfg<TX, TY>;
    constexpr int PL = Cfg::PL;
    const bool with_b = u >= 0;
    unsigned long long* bar = bars + ((u + 1) & 3);
    double* da = sm + Cfg::RING_A + ((u + 1) & 3) * (Cfg::NA * PL);
    double* db = sm + Cfg::RING_B + (u & 1) * (Cfg::NB * PL);
    dr_mbar_expect_tx(bar, with_b ? Cfg::BYTES_A + Cfg::BYTES_B : Cfg::BYTES_A);
#pragma unroll
    for (int f = 0; f < 3; ++f) dr_tma_load_3d(da + f * PL, T.m + f, bar, x0, y0, m + 1, T.l2_hint);
    dr_bulk_load_1d(da + 3 * PL, codesrc + codestride * (m + TB2_KLO), PL * sizeof(double), bar);
    if (with_b) {
#pragma unroll
        for (int f = 0; f < 4; ++f) dr_tma_load_3d(db + f * PL, T.m + 3 + f, bar, x0, y0, m, T.l2_hint);
        dr_tma_load_3d(db + 4 * PL, T.m + 7, bar, x0, y0, m + 1, T.l2_hint);
        dr_tma_load_3d(db + 5 * PL, T.m + 8, bar, x0, y0, m + 1, T.l2_hint);
    }
}

// output: the 9 fields of the new state sit at a constant stride (fs doubles) in the workspace, in the order of dr_layout.cuh
// (vx vy vz sxx syy szz tyz txz txy); col = this thread's node column in field 0.  One pointer instead of nine.
struct DrTb2Out { double* col; long long fs; };

// step t of the march: first-iteration layer k = kb - 2 + t, second-iteration layer k2 = k - 2.  Q = t & 3 is a template
// parameter so that every shared-memory offset (ring slots, parity buffers) is a compile-time constant relative to the
// thread's own address: the compiler can then interleave the four stages freely.
// code2: in = stencil code of layer k-2 (stored by step t-2, same parity), out = that of layer k.
template <int RES, int NIT, int TX, int TY, bool BND, int Q>
__device__ __forceinline__ void dr_tb2_step(const DrTb2Batch& TB, const DrLayout& L, const DrPT& P, const DrTb2Maps& T, const DrTb2Out& g,
                                            double* sm, const double* tab, const unsigned long long* codesrc, const long long codestride,
                                            unsigned long long* bars, const int s, const int t, const int k,
                                            const int kb, const int ke, const int i, const int j, const int x0, const int y0,
                                            const bool producer, const bool in1, const bool row1, const bool row2, const bool in2,
                                            const DrFace5& fc, DrFace5& fn, const DrFace5& gc, DrFace5& gn,
                                            unsigned long long& code2, double& rmax, bool& rnan) {
    using Cfg = DrTb2Cfg<TX, TY>;
    constexpr int PL = Cfg::PL;
    constexpr int PAR = Q & 1;
    const int nx = L.nx, ny = L.ny, nz = L.nz;
    const long long sz = L.sz;
    const int ke1 = ke + (NIT == 2 ? 1 : 0);                  // one past the last first-iteration layer
    const int k2 = k - 2;
    const bool act1 = k < ke1;                                // uniform over the CTA
    const bool act2 = (NIT == 2) && k2 >= kb - 1;             // uniform
    double* X1p = sm + Cfg::X1 + PAR * (Y_COUNT * PL) + s;    // on entry: first-iteration stresses of layer k-2
    double* V1c = sm + Cfg::V1 + PAR * (3 * PL) + s;          // first-iteration velocities of layer k-2; B1 puts layer k here
    const double* V1n = sm + Cfg::V1 + (1 - PAR) * (3 * PL) + s;     // ... of layer k-1
    double* X2p = sm + Cfg::X2 + s;
    const unsigned long long c2 = code2;                      // layer k-2

    // ================= phase alpha =================
    DrStress6 r2;                                             // second-iteration stresses, own node (TB2_REREAD 0)
    r2.sxx = r2.syy = r2.szz = r2.txy = r2.txz = r2.tyz = 0.0;
    // second-iteration stresses are read by B2 at the inner rows and their +-1 neighbours: rows 1 .. TY-2 (a warp is a row)
    if (act2 && (!TB2_SKIPA2 || row1)) {
        DrStress6 o;
        o.sxx = X1p[Y_SXX * PL]; o.syy = X1p[Y_SYY * PL]; o.szz = X1p[Y_SZZ * PL];
        o.txy = X1p[Y_TXY * PL]; o.txz = X1p[Y_TXZ * PL]; o.tyz = X1p[Y_TYZ * PL];
        double lam2, g22;
        dr_tab_lg(TB, tab, dr_code_off(c2, 0), lam2, g22);
        const DrStress6 m2 = dr_tb2_stress<BND>(P, nx, ny, nz, i, j, k2, lam2, g22,
                                TB2_TAB(TB2_S_ES, dr_code_off(c2, 1)), TB2_TAB(TB2_S_ES, dr_code_off(c2, 2)), TB2_TAB(TB2_S_ES, dr_code_off(c2, 3)),
                                V1c[0 * PL], V1c[1 * PL], V1c[2 * PL], V1c[0 * PL + 1], V1c[1 * PL + TX], V1c[0 * PL - TX], V1c[1 * PL - 1],
                                V1n[0 * PL], V1n[1 * PL], V1n[2 * PL], V1n[2 * PL - 1], V1n[2 * PL - TX], o);
        X2p[Z_SXX * PL] = m2.sxx; X2p[Z_SYY * PL] = m2.syy; X2p[Z_TXY * PL] = m2.txy;
        X2p[Z_TXZ * PL] = m2.txz; X2p[Z_TYZ * PL] = m2.tyz;
        gn.txz = m2.txz; gn.tyz = m2.tyz; gn.szz = m2.szz;
        if (!TB2_REREAD) r2 = m2;
    }
    DrStress6 m1;                                             // first-iteration stresses (own node)
    double vxc = 0.0, vyc = 0.0, vzc = 0.0;
    unsigned long long c1 = 0ull;
    if (act1) {
        const int qa = TB2_UNROLL4 ? Q : (t & 3);
        const double* Ac = sm + Cfg::RING_A + qa * (Cfg::NA * PL) + s;                 // layer k
        const double* An = sm + Cfg::RING_A + ((qa + 1) & 3) * (Cfg::NA * PL) + s;     // layer k+1
        const double* Bs = sm + Cfg::RING_B + PAR * (Cfg::NB * PL) + s;                // old stresses of this step
        c1 = *reinterpret_cast<const unsigned long long*>(Ac + 3 * PL);
        vxc = Ac[0 * PL]; vyc = Ac[1 * PL]; vzc = Ac[2 * PL];
        DrStress6 o;
        o.sxx = Bs[0 * PL]; o.syy = Bs[1 * PL]; o.szz = Bs[2 * PL]; o.txy = Bs[3 * PL]; o.txz = Bs[4 * PL]; o.tyz = Bs[5 * PL];
        double lam1, g21;
        dr_tab_lg(TB, tab, dr_code_off(c1, 0), lam1, g21);
        m1 = dr_tb2_stress<BND>(P, nx, ny, nz, i, j, k, lam1, g21,
                                TB2_TAB(TB2_S_ES, dr_code_off(c1, 1)), TB2_TAB(TB2_S_ES, dr_code_off(c1, 2)), TB2_TAB(TB2_S_ES, dr_code_off(c1, 3)),
                                vxc, vyc, vzc, Ac[0 * PL + 1], Ac[1 * PL + TX], Ac[0 * PL - TX], Ac[1 * PL - 1],
                                An[0 * PL], An[1 * PL], An[2 * PL], An[2 * PL - 1], An[2 * PL - TX], o);
        // X1p held layer k-2 (read above by this same thread): now layer k
        X1p[Y_SXX * PL] = m1.sxx; X1p[Y_SYY * PL] = m1.syy; X1p[Y_TXY * PL] = m1.txy;
        X1p[Y_TXZ * PL] = m1.txz; X1p[Y_TYZ * PL] = m1.tyz;
        if (NIT == 2) X1p[Y_SZZ * PL] = m1.szz;
        fn.txz = m1.txz; fn.tyz = m1.tyz; fn.szz = m1.szz;
        code2 = c1;
    }
    __syncthreads();

    // ---- every thread is done with ring-A layer k-1 (since the previous step) and with this step's ring-B set: their
    // slots take group t+2 = layer k+3 and the stress set of step t+2, one and a half steps ahead of need
    if (producer && k + 2 < ke1)
        dr_tb2_issue_group<TX, TY>(T, bars, sm, codesrc, codestride, x0, y0, t + 2, k + 3);
    // ---- the group of the next step (issued one step ago)
    if (k + 1 < ke1) dr_mbar_wait(bars + (((TB2_UNROLL4 ? Q : t) + 2) & 3), ((t + 2) >> 2) & 1);

    // ================= phase beta =================
    if (act2 && row2) {
        const double* Z = X2p;
        gn.txz_r = Z[Z_TXZ * PL + 1]; gn.tyz_u = Z[Z_TYZ * PL + TX];       // +x / +y neighbours on face k2+1, for the next step
        if (in2 && k2 >= kb) {
            // own second-iteration stresses come back from the exchange planes (not held in registers across the barrier)
            const double msxx = TB2_REREAD ? Z[Z_SXX * PL] : r2.sxx, msyy = TB2_REREAD ? Z[Z_SYY * PL] : r2.syy, mtxy = TB2_REREAD ? Z[Z_TXY * PL] : r2.txy;
            double* const po = g.col + sz * k2;
            const bool ck = k2 < nz;
            const bool ci = !BND || i < nx, cj = !BND || j < ny;
            if (ck) {
                if (cj) {                           // v_x at (i, j+1/2, k2+1/2)
                    const double Fx = (msxx - Z[Z_SXX * PL - 1]) + (Z[Z_TXY * PL + TX] - mtxy) + (gn.txz - gc.txz);
                    po[F_VX * g.fs] = dr_tb2_vel<RES>(V1c[0 * PL], Fx, TB, tab, dr_code_off(c2, 4), rmax, rnan);
                    po[F_TXZ * g.fs] = gc.txz;
                }
                if (ci) {                           // v_y at (i+1/2, j, k2+1/2)
                    const double Fy = (Z[Z_TXY * PL + 1] - mtxy) + (msyy - Z[Z_SYY * PL - TX]) + (gn.tyz - gc.tyz);
                    po[F_VY * g.fs] = dr_tb2_vel<RES>(V1c[1 * PL], Fy, TB, tab, dr_code_off(c2, 5), rmax, rnan);
                    po[F_TYZ * g.fs] = gc.tyz;
                }
                po[F_TXY * g.fs] = mtxy;
                if (ci && cj) { po[F_SXX * g.fs] = msxx; po[F_SYY * g.fs] = msyy; po[F_SZZ * g.fs] = gn.szz; }
            } else {                                // k2 == nz: only the top faces
                if (cj) po[F_TXZ * g.fs] = gc.txz;
                if (ci) po[F_TYZ * g.fs] = gc.tyz;
            }
            if (ci && cj) {                         // v_z at (i+1/2, j+1/2, k2)
                const double Fz = (gc.txz_r - gc.txz) + (gc.tyz_u - gc.tyz) + (gn.szz - gc.szz);
                po[F_VZ * g.fs] = dr_tb2_vel<RES>(V1c[2 * PL], Fz, TB, tab, dr_code_off(c2, 6), rmax, rnan);
            }
        }
    }
    if (act1) {
        const double* Y = X1p;
        double nvx = vxc, nvy = vyc, nvz = vzc;
        double r1 = 0.0; bool n1 = false;                    // the first iteration of a pair is never a check iteration
        if (in1) {
            fn.txz_r = Y[Y_TXZ * PL + 1]; fn.tyz_u = Y[Y_TYZ * PL + TX];
            const double Fx = (m1.sxx - Y[Y_SXX * PL - 1]) + (Y[Y_TXY * PL + TX] - m1.txy) + (m1.txz - fc.txz);
            const double Fy = (Y[Y_TXY * PL + 1] - m1.txy) + (m1.syy - Y[Y_SYY * PL - TX]) + (m1.tyz - fc.tyz);
            const double Fz = (fc.txz_r - fc.txz) + (fc.tyz_u - fc.tyz) + (m1.szz - fc.szz);
            if (NIT == 2) {
                nvx = dr_tb2_vel<0>(vxc, Fx, TB, tab, dr_code_off(c1, 4), r1, n1);
                nvy = dr_tb2_vel<0>(vyc, Fy, TB, tab, dr_code_off(c1, 5), r1, n1);
                nvz = dr_tb2_vel<0>(vzc, Fz, TB, tab, dr_code_off(c1, 6), r1, n1);
            } else if (row2 && in2 && k >= kb) {    // NIT == 1: a plain one-iteration sweep on the same geometry
                double* const po = g.col + sz * k;
                const bool ck = k < nz;
                const bool ci = !BND || i < nx, cj = !BND || j < ny;
                if (ck) {
                    if (cj) { po[F_VX * g.fs] = dr_tb2_vel<RES>(vxc, Fx, TB, tab, dr_code_off(c1, 4), rmax, rnan); po[F_TXZ * g.fs] = fc.txz; }
                    if (ci) { po[F_VY * g.fs] = dr_tb2_vel<RES>(vyc, Fy, TB, tab, dr_code_off(c1, 5), rmax, rnan); po[F_TYZ * g.fs] = fc.tyz; }
                    po[F_TXY * g.fs] = m1.txy;
                    if (ci && cj) { po[F_SXX * g.fs] = m1.sxx; po[F_SYY * g.fs] = m1.syy; po[F_SZZ * g.fs] = m1.szz; }
                } else {
                    if (cj) po[F_TXZ * g.fs] = fc.txz;
                    if (ci) po[F_TYZ * g.fs] = fc.tyz;
                }
                if (ci && cj) po[F_VZ * g.fs] = dr_tb2_vel<RES>(vzc, Fz, TB, tab, dr_code_off(c1, 6), rmax, rnan);
            }
        }
        if (NIT == 2) { V1c[0 * PL] = nvx; V1c[1 * PL] = nvy; V1c[2 * PL] = nvz; }   // layer k replaces layer k-2 (read above)
    }
    if (NIT == 2) __syncthreads();
}

template <int RES, int NIT, int TX, int TY, bool BND>
__device__ __forceinline__ void dr_tb2_march(const DrTb2Batch& TB, const DrLayout& L, const DrPT& P, const DrTb2Maps& T, const DrTb2Out& g,
                                             double* sm, const double* tab, const unsigned long long* codesrc, const long long codestride,
                                             unsigned long long* bars, const int s, const int kb, const int ke,
                                             const int i, const int j, const int x0, const int y0,
                                             const bool producer, const bool in1, const bool row1, const bool row2, const bool in2, double& rmax, bool& rnan) {
    DrFace5 fa, fb, ga, gb;
    fa.txz = fa.tyz = fa.szz = fa.txz_r = fa.tyz_u = 0.0;
    fb = fa; ga = fa; gb = fa;
    unsigned long long ca = 0ull, cb = 0ull;
    const int klast = ke + (NIT == 2 ? 1 : -1);               // last step: second iteration of layer ke-1
    int k = kb - 2;
#define DR_TB2_STEP(Q_, FC, FN, GC, GN, CC) \
    dr_tb2_step<RES, NIT, TX, TY, BND, Q_>(TB, L, P, T, g, sm, tab, codesrc, codestride, bars, s, t + Q_, k + Q_, kb, ke, i, j, x0, y0, producer, in1, row1, row2, in2, FC, FN, GC, GN, CC, rmax, rnan)
#if TB2_UNROLL4
    for (int t = 0; k <= klast; t += 4, k += 4) {
        DR_TB2_STEP(0, fa, fb, ga, gb, ca);
        if (k + 1 <= klast) DR_TB2_STEP(1, fb, fa, gb, ga, cb);
        if (k + 2 <= klast) DR_TB2_STEP(2, fa, fb, ga, gb, ca);
        if (k + 3 <= klast) DR_TB2_STEP(3, fb, fa, gb, ga, cb);
    }
#else
    for (int t = 0; k <= klast; t += 2, k += 2) {
        DR_TB2_STEP(0, fa, fb, ga, gb, ca);
        if (k + 1 <= klast) DR_TB2_STEP(1, fb, fa, gb, ga, cb);
    }
#endif
#undef DR_TB2_STEP
}

// NIT = 2: two PT iterations per launch (RES: the residual max-norm of the SECOND one); NIT = 1: one iteration on the same
// geometry and tables (kept for A/B checks of the coded path against k_pt_tma).
template <int RES, int NIT, int TX, int TY>
__global__ void __launch_bounds__(TX * TY, 1)
k_pt_tb2(const __grid_constant__ DrTb2Batch TB, DrLayout L, int lz) {
    extern __shared__ __align__(1024) double sm[];
    __shared__ __align__(8) unsigned long long bars[4];
#if TB2_CTAB
    const double* const tab = nullptr;                        // tables: TB.dtab, read with LDC
#else
    __shared__ __align__(16) double tab[RES ? 1280 : 1024];
#endif
    using Cfg = DrTb2Cfg<TX, TY>;
    constexpr int PL = Cfg::PL;
    const int nx = L.nx, ny = L.ny, nz = L.nz;
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int slot = blockIdx.z / TB.nchunks, chunk = blockIdx.z - slot * TB.nchunks;
    const DrPT& P = TB.P[slot];
    DrTb2Maps T;
    T.m = TB.m[slot]; T.l2_hint = TB.l2_hint;
    // node of thread (0,0): ib is odd so that the TMA box starts on an even element (16-byte aligned, DR_OX is odd)
    const int ib = blockIdx.x * (TX - 4) - 3, jb = blockIdx.y * (TY - 4) - 2;
    const int i = ib + tx, j = jb + ty;
    const int kb = chunk * lz;
    const int ke = min(kb + lz, nz + 1);
    const int x0 = DR_OX + ib, y0 = jb + 1;                  // box origin in padded-field coordinates (z = layer + 1)
    const long long codestride = (long long)TB.gx * TB.gy * PL;
    const unsigned long long* codesrc = TB.codes + ((long long)blockIdx.y * TB.gx + blockIdx.x) * PL;
    const int s = ty * TX + tx;
    // derived tables (see TB2_S_*): the products that do not change from one iteration to the next
#if !TB2_CTAB
    {
        const double thh = P.theta * P.inv_h, cvh = P.c2t * P.inv_h;
        for (int e = s; e < 256; e += TX * TY) {
            const double Kv = TB.tabs[TB2_TAB_K + e], Gv = TB.tabs[TB2_TAB_G + e], Rv = TB.tabs[TB2_TAB_R + e];
            tab[TB2_LG128 ? 2 * e : TB2_S_LAM + e] = fma(-(2.0 / 3.0), Gv, Kv);
            tab[TB2_LG128 ? 2 * e + 1 : TB2_S_G2 + e] = 2.0 * Gv;
            tab[TB2_S_ES + e] = thh * TB.tabs[TB2_TAB_E + e];
            tab[TB2_S_CV + e] = cvh * Rv;
            if (RES) tab[TB2_S_RH + e] = Rv;
        }
    }
#endif
    const bool producer = (tx == 0 && ty == 0);
    const bool in1 = tx >= 1 && tx <= TX - 2 && ty >= 1 && ty <= TY - 2;
    const bool row1 = ty >= 1 && ty <= TY - 2;
    const bool row2 = ty >= 2 && ty <= TY - 3;
    const bool in2 = tx >= 2 && tx <= TX - 3 && i >= 0 && i <= nx && j <= ny;

    if (producer) {
#pragma unroll
        for (int b = 0; b < 4; ++b) dr_mbar_init(bars + b, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        // prologue: group -1 = layer kb-2, groups 0 and 1 = layers kb-1, kb with the stress sets of steps 0 and 1
        dr_tb2_issue_group<TX, TY>(T, bars, sm, codesrc, codestride, x0, y0, -1, kb - 2);
        dr_tb2_issue_group<TX, TY>(T, bars, sm, codesrc, codestride, x0, y0, 0, kb - 1);
        dr_tb2_issue_group<TX, TY>(T, bars, sm, codesrc, codestride, x0, y0, 1, kb);
    }
    __syncthreads();                                          // barrier init and tables visible
    dr_mbar_wait(bars + 0, 0);
    dr_mbar_wait(bars + 1, 0);

    DrTb2Out g;
    g.col = TB.out[slot] + (L.origin + min(max(i, 0), nx + 1) + L.sy * min(max(j, 0), ny + 1));
    g.fs = TB.fs;
    double rmax = 0.0;
    bool rnan = false;
    // extended tile free of boundary nodes?
    const bool interior = ib >= 1 && ib + TX - 1 <= nx - 1 && jb >= 1 && jb + TY - 1 <= ny - 1;
    if (interior) dr_tb2_march<RES, NIT, TX, TY, false>(TB, L, P, T, g, sm, tab, codesrc, codestride, bars, s, kb, ke, i, j, x0, y0, producer, in1, row1, row2, in2, rmax, rnan);
    else          dr_tb2_march<RES, NIT, TX, TY, true>(TB, L, P, T, g, sm, tab, codesrc, codestride, bars, s, kb, ke, i, j, x0, y0, producer, in1, row1, row2, in2, rmax, rnan);

    if (RES) {
        __shared__ unsigned long long smr[32];
        unsigned long long b = rnan ? 0x7ff8000000000000ull : (unsigned long long)__double_as_longlong(rmax * (P.inv_h * P.res_scale));
        __syncthreads();
        b = dr_block_max_bits(b, smr);
        if (tx == 0 && ty == 0 && b != 0ull) atomicMax(TB.res[slot], b);
    }
}

// =====================================================================================================================
// Stencil codes and tables (once per image / DR_GAVG / DR_VOID_REL)
// =====================================================================================================================
#define DR_TAB_EMPTY 0xffffffffffffffffull      // a NaN pattern: never a table value

__device__ __forceinline__ unsigned dr_tab_hash(unsigned long long b) { return (unsigned)((b * 0x9E3779B97F4A7C15ull) >> 56); }

// insert (or find) a value in a 256-slot open-addressing table; -1 when the table is full of other values
__device__ __forceinline__ int dr_tab_insert(unsigned long long* keys, unsigned long long b) {
    const unsigned h = dr_tab_hash(b);
    for (int p = 0; p < 256; ++p) {
        const int slot = (h + p) & 255;
        unsigned long long o = keys[slot];
        if (o == DR_TAB_EMPTY) o = atomicCAS(keys + slot, DR_TAB_EMPTY, b);
        if (o == DR_TAB_EMPTY || o == b) return slot;
    }
    return -1;
}
__device__ __forceinline__ int dr_tab_find(const unsigned long long* keys, unsigned long long b) {
    const unsigned h = dr_tab_hash(b);
    for (int p = 0; p < 256; ++p) {
        const int slot = (h + p) & 255;
        if (keys[slot] == b) return slot;
        if (keys[slot] == DR_TAB_EMPTY) return -1;
    }
    return -1;
}

// the seven moduli-only quantities of node column (i,j), layer k, exactly as k_pt_tma evaluates them on the fly
// (dr_edge_mean_fast in the same argument order, hc = fma(4/3, G, K), dr_rcp); indices are clamped into the padded box,
// whose halo is replicate-padded (Reading R4), so out-of-domain positions give harmless finite values
struct DrNodeVals { double exy, exz, eyz, rx, ry, rz; };

template <int GAVG>
__device__ __forceinline__ DrNodeVals dr_code_values(const DrLayout& L, const double* __restrict__ Kp, const double* __restrict__ Gp, int i, int j, int k) {
    const int nx = L.nx, ny = L.ny, nz = L.nz;
    auto Q = [&](int a, int b, int c) -> long long {
        return L.origin + min(max(a, -1), nx) + L.sy * min(max(b, -1), ny) + L.sz * min(max(c, -1), nz);
    };
    auto Gv = [&](int a, int b, int c) -> double { return Gp[Q(a, b, c)]; };
    auto Hv = [&](int a, int b, int c) -> double { const long long q = Q(a, b, c); return fma(4.0 / 3.0, Gp[q], Kp[q]); };
    auto Exy = [&](int a, int b, int c) -> double { return dr_edge_mean_fast<GAVG>(Gv(a - 1, b - 1, c), Gv(a, b - 1, c), Gv(a - 1, b, c), Gv(a, b, c)); };
    auto Exz = [&](int a, int b, int c) -> double { return dr_edge_mean_fast<GAVG>(Gv(a - 1, b, c - 1), Gv(a, b, c - 1), Gv(a - 1, b, c), Gv(a, b, c)); };   // face c
    auto Eyz = [&](int a, int b, int c) -> double { return dr_edge_mean_fast<GAVG>(Gv(a, b - 1, c - 1), Gv(a, b, c - 1), Gv(a, b - 1, c), Gv(a, b, c)); };   // face c
    DrNodeVals v;
    const double exy = Exy(i, j, k), exz0 = Exz(i, j, k), exz1 = Exz(i, j, k + 1), eyz0 = Eyz(i, j, k), eyz1 = Eyz(i, j, k + 1);
    v.exy = exy; v.exz = exz1; v.eyz = eyz1;
    const double hc = Hv(i, j, k);
    const bool ci = i >= 0 && i < nx, cj = j >= 0 && j < ny, ck = k >= 0 && k < nz;
    v.rx = v.ry = v.rz = 0.0;
    if (i >= 1 && i <= nx - 1 && cj && ck) {            // interior v_x node (walls keep their value, SURVEY O6 rule N)
        const double Hn = dr_max(dr_max(dr_max(Hv(i - 1, j, k), hc), dr_max(exy, Exy(i, j + 1, k))), dr_max(exz0, exz1));
        if (Hn > 0.0) v.rx = dr_rcp(Hn);
    }
    if (j >= 1 && j <= ny - 1 && ci && ck) {
        const double Hn = dr_max(dr_max(dr_max(Hv(i, j - 1, k), hc), dr_max(exy, Exy(i + 1, j, k))), dr_max(eyz0, eyz1));
        if (Hn > 0.0) v.ry = dr_rcp(Hn);
    }
    if (k >= 1 && k <= nz - 1 && ci && cj) {
        const double Hn = dr_max(dr_max(dr_max(Hv(i, j, k - 1), hc), dr_max(exz0, Exz(i + 1, j, k))), dr_max(eyz0, Eyz(i, j + 1, k)));
        if (Hn > 0.0) v.rz = dr_rcp(Hn);
    }
    return v;
}

// PASS 0: insert the values of every coded position into the edge / node tables (flags |= 8 on overflow)
// PASS 1: look them up and write the code words (flags |= 16 on a miss, which cannot happen after a complete pass 0)
// grid (gx, gy, nz + KLO + KHI), block (TX, TY); K0p/G0p = unclamped padded moduli (keys of the cell palette)
template <int GAVG, int PASS>
__global__ void k_code_build(DrLayout L, const double* __restrict__ Kp, const double* __restrict__ Gp,
                             const double* __restrict__ K0p, const double* __restrict__ G0p,
                             const unsigned long long* __restrict__ palK, const unsigned long long* __restrict__ palG,
                             unsigned long long* ekeys, unsigned long long* rkeys,
                             unsigned long long* __restrict__ codes, unsigned int* flags) {
    const int TX = blockDim.x, TY = blockDim.y;
    const int i = blockIdx.x * (TX - 4) - 3 + threadIdx.x;
    const int j = blockIdx.y * (TY - 4) - 2 + threadIdx.y;
    const int k = (int)blockIdx.z - TB2_KLO;
    const DrNodeVals v = dr_code_values<GAVG>(L, Kp, Gp, i, j, k);
    const unsigned long long b[6] = {(unsigned long long)__double_as_longlong(v.exy), (unsigned long long)__double_as_longlong(v.exz),
                                     (unsigned long long)__double_as_longlong(v.eyz), (unsigned long long)__double_as_longlong(v.rx),
                                     (unsigned long long)__double_as_longlong(v.ry), (unsigned long long)__double_as_longlong(v.rz)};
    if (PASS == 0) {
        if (*((volatile unsigned int*)flags) & 8u) return;
        bool bad = false;
#pragma unroll
        for (int e = 0; e < 3; ++e) bad |= dr_tab_insert(ekeys, b[e]) < 0;
#pragma unroll
        for (int e = 3; e < 6; ++e) bad |= dr_tab_insert(rkeys, b[e]) < 0;
        if (bad) atomicOr(flags, 8u);
        return;
    }
    const long long q = L.origin + min(max(i, -1), L.nx) + L.sy * min(max(j, -1), L.ny) + L.sz * min(max(k, -1), L.nz);
    const int cell = dr_pal_find(palK, palG, (unsigned long long)__double_as_longlong(K0p[q]), (unsigned long long)__double_as_longlong(G0p[q]));
    unsigned long long code = (unsigned long long)(cell < 0 ? 0 : cell);
    bool miss = cell < 0;
#pragma unroll
    for (int e = 0; e < 6; ++e) {
        const int id = dr_tab_find(e < 3 ? ekeys : rkeys, b[e]);
        miss |= id < 0;
        code |= (unsigned long long)(id < 0 ? 0 : id) << (8 * (e + 1));
    }
    if (miss) atomicOr(flags, 16u);
    const size_t blk = ((size_t)blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
    codes[blk * (size_t)(TX * TY) + threadIdx.y * TX + threadIdx.x] = code;
}

// table values from the keys: tabs[0..511] = cell palette K, G (copied from pal), tabs[512..767] = E, tabs[768..1023] = R
__global__ void k_code_tables(const double* __restrict__ pal, const unsigned long long* __restrict__ ekeys,
                              const unsigned long long* __restrict__ rkeys, double* __restrict__ tabs) {
    const int e = threadIdx.x;
    tabs[TB2_TAB_K + e] = pal[e];
    tabs[TB2_TAB_G + e] = pal[256 + e];
    tabs[TB2_TAB_E + e] = ekeys[e] == DR_TAB_EMPTY ? 0.0 : __longlong_as_double((long long)ekeys[e]);
    tabs[TB2_TAB_R + e] = rkeys[e] == DR_TAB_EMPTY ? 0.0 : __longlong_as_double((long long)rkeys[e]);
}
