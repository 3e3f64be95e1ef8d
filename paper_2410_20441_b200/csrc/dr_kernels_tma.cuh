// dr_kernels_tma.cuh -- fused PT iteration with TMA halo staging (SURVEY 8(a) row a2+a3, the graded kernel).
//
// Same arithmetic and the same 2.5-D z-march as dr_kernels_fused.cuh (one launch = one PT iteration, stress
// update Eq. 12-13 P:90-94 then velocity update Eq. 11 P:86, 160 B compulsory per voxel-iteration), but the
// inputs never pass through registers on their way in: one elected thread issues cp.async.bulk.tensor (TMA)
// copies of the (TX x TY x 1) extended tile of every field, several z layers ahead, into shared-memory rings;
// completion is signalled on mbarriers.  This decouples the bytes in flight (about two layers = 90 KB per SM)
// from the register file, which is what limits the LDG version.
//
//   ring A (4 slots): vx vy vz G of one layer            -- layer k ("c") and k+1 ("n") are read at step k
//   ring B (3 slots): K sxx syy szz txy of layer m-1 and txz tyz of face m   -- the set m = k+1 is read at step k
//   batch m = ring A layer m + ring B set m, issued together right after the second barrier of step m-4
//
// Out-of-range parts of a box (beyond the padded field) are zero-filled by the TMA unit; the halo ring inside
// the padded field holds zeros (state) or replicate-padded moduli, so no index clamping is needed.
#pragma once
#include <cuda.h>
#include "dr_kernels_fused.cuh"

#define DR_TMA_SA 4
#define DR_TMA_SB 3
#define DR_TMA_NA 4      // fields per ring-A slot (3 with the palette: no G plane)
#define DR_TMA_NB 7      // fields per ring-B slot (6 with the palette: no K plane)

// PAL = 1 (palette path): images with at most 256 distinct (K,G) pairs -- every segmented rock image -- keep a uint8
// phase id per cell; the kernel stages the ids of its extended tile instead of the two fp64 modulus boxes and looks K, G
// up in a 256-entry table in shared memory.  Same arithmetic on the same values, about 15 B less HBM traffic per
// voxel-iteration and 96 fewer 128-byte lines through L2 per CTA step.  The ids are stored TILE-BLOCKED: for every
// (tile, layer) the TX*TY ids of the extended tile are contiguous (halo ids duplicated, they never change), so one
// plain 1-D cp.async.bulk of 512 B brings them; as a 16-row tensor box they cost as much as a whole fp64 box.
// tensor maps of one launch: 0..3 = vx vy vz G, 4..10 = K sxx syy szz txy txz tyz (old state + moduli)
struct DrTmaps {
    CUtensorMap m[DR_TMA_NA + DR_TMA_NB];
    const unsigned char* ids;       // [nz+3][gy][gx][TY][TX] phase ids (layer -1 first)
    const double* pal;              // K[256], G[256]
    int gx, gy;                     // tiles in x and y
    unsigned long long l2_hint;
};

template <int TX, int TY, int PAL = 0>
struct DrTmaCfg {
    static constexpr int PL = TX * TY;                               // doubles per dense plane
    static constexpr int NA = PAL ? DR_TMA_NA - 1 : DR_TMA_NA;       // planes per ring-A slot
    static constexpr int NB = PAL ? DR_TMA_NB - 1 : DR_TMA_NB;       // planes per ring-B slot
    static constexpr int BK = PAL ? 0 : 1;                           // first state plane of a ring-B slot (K sits before it)
    static constexpr int FRONT = 128;                                // pad (doubles) before the first plane
    static constexpr int RING_A = FRONT;                             // [SA][NA][PL]
    static constexpr int RING_B = RING_A + DR_TMA_SA * NA * PL;      // [SB][NB][PL]
    static constexpr int XCH = RING_B + DR_TMA_SB * NB * PL;         // exchange planes
    static constexpr int END = XCH + 13 * PL;
    static constexpr size_t SMEM = (size_t)(END + 64) * sizeof(double);
    static constexpr unsigned BYTES_A = NA * PL * sizeof(double);
    static constexpr unsigned BYTES_B = NB * PL * sizeof(double);
};

__device__ __forceinline__ unsigned dr_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void dr_mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(dr_smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void dr_mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(dr_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void dr_mbar_wait(unsigned long long* bar, unsigned parity) {
    asm volatile(
        "{\n\t.reg .pred P1;\n\t"
        "DR_WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
        "@P1 bra DR_DONE_%=;\n\t"
        "bra DR_WAIT_%=;\n\t"
        "DR_DONE_%=:\n\t}"
        ::"r"(dr_smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void dr_tma_load_3d(void* dst, const CUtensorMap* map, unsigned long long* bar, int x, int y, int z,
                                               unsigned long long hint) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%3, %4, %5}], [%2], %6;"
        ::"r"(dr_smem_u32(dst)), "l"((unsigned long long)map), "r"(dr_smem_u32(bar)), "r"(x), "r"(y), "r"(z), "l"(hint) : "memory");
}

__device__ __forceinline__ void dr_bulk_load_1d(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dr_smem_u32(dst)), "l"((unsigned long long)src), "r"(bytes), "r"(dr_smem_u32(bar)) : "memory");
}

// one batch: ring-A fields of layer m (z = m+1 in the padded box) and, if with_b, the ring-B set m:
//   FORM 0: K, sigma_xx, sigma_yy, sigma_zz, tau_xy of layer m-1 and tau_xz, tau_yz of face m
//   FORM 1: K, w_x, w_y, w_z of layer m-1 (w lives in the sigma_aa slots of the state buffer)
template <int FORM, int PAL, int TX, int TY>
__device__ __forceinline__ void dr_tma_issue_batch(const DrTmaps& T, unsigned long long* bar, double* da, double* db,
                                                   unsigned char* idd, const unsigned char* idsrc, long long idstride,
                                                   int x0, int y0, int m, bool with_b) {
    constexpr int PL = TX * TY;
    constexpr unsigned BA = 3 * PL * sizeof(double) + (PAL ? PL : PL * sizeof(double));
    constexpr unsigned BB = ((FORM ? 3 : 6) + (PAL ? 0 : 1)) * PL * sizeof(double);
    constexpr int BK = PAL ? 0 : 1;
    dr_mbar_expect_tx(bar, with_b ? BA + BB : BA);
#pragma unroll
    for (int f = 0; f < 3; ++f) dr_tma_load_3d(da + f * PL, &T.m[f], bar, x0, y0, m + 1, T.l2_hint);
    if (PAL) dr_bulk_load_1d(idd, idsrc + idstride * (m + 1), PL, bar);
    else     dr_tma_load_3d(da + 3 * PL, &T.m[3], bar, x0, y0, m + 1, T.l2_hint);
    if (with_b) {
        if (!PAL) dr_tma_load_3d(db, &T.m[4], bar, x0, y0, m, T.l2_hint);                   // K of layer m-1
#pragma unroll
        for (int f = 0; f < (FORM ? 3 : 4); ++f) dr_tma_load_3d(db + (BK + f) * PL, &T.m[5 + f], bar, x0, y0, m, T.l2_hint);
        if (!FORM) {
            dr_tma_load_3d(db + (BK + 4) * PL, &T.m[9], bar, x0, y0, m + 1, T.l2_hint);
            dr_tma_load_3d(db + (BK + 5) * PL, &T.m[10], bar, x0, y0, m + 1, T.l2_hint);
        }
    }
}

// new values a thread carries from one step to the next (registers): its own tau / edge moduli on the face
// between the layers, sigma_zz and H of the layer below, and the +x / +y neighbours' face values
struct DrCarry { double txz, tyz, gxz, gyz, szz, hc, txz_r, tyz_u, gxz_r, gyz_u; };

// exchange planes (doubles, relative to XCH), double-buffered by step parity: [2][9][PL]
enum { X_SXX = 0, X_SYY, X_TXY, X_HC, X_GXY, X_TXZ, X_TYZ, X_GXZ, X_GYZ, X_COUNT };

template <int TX, int TY, int PAL = 0>
struct DrTmaCfg2 : DrTmaCfg<TX, TY, PAL> {
    using B = DrTmaCfg<TX, TY, PAL>;
    static constexpr int END2 = B::XCH + 2 * X_COUNT * B::PL;
    static constexpr size_t SMEM2 = (size_t)(END2 + 64) * sizeof(double);
};

template <int GAVG, int RES, int FORM, int PAL, int TX, int TY, bool BND, int PAR>
__device__ __forceinline__ void dr_tma_step(const DrLayout& L, const DrPT& P, const DrTmaps& T, const DrFusedPtrs& g,
                                            double* sm, unsigned char* idr, const double* pal, const unsigned char* idsrc,
                                            const long long idstride,
                                            unsigned long long* bars, const int s, const int t, const int k,
                                            const int kb, const int ke, const bool store, const int i, const int j,
                                            const int x0, const int y0, const bool producer, const bool midrow, const bool inner,
                                            const DrCarry& fc, DrCarry& fn, double& rmax, bool& rnan) {
    using Cfg = DrTmaCfg2<TX, TY, PAL>;
    constexpr int PL = Cfg::PL, BK = Cfg::BK;
    const int nx = L.nx, ny = L.ny, nz = L.nz;
    const long long sz = L.sz;
    const double h = P.h, ih = P.inv_h, th = P.theta, ri = P.rinv, c2t = P.c2t;
    const double* Ac = sm + Cfg::RING_A + (t & 3) * (Cfg::NA * PL) + s;            // layer k
    const double* An = sm + Cfg::RING_A + ((t + 1) & 3) * (Cfg::NA * PL) + s;      // layer k+1
    const double* Bs = sm + Cfg::RING_B + (t % 3) * (Cfg::NB * PL) + s;            // set k+1
    const unsigned char* Ic = idr + (t & 3) * PL + s;                               // phase ids of layer k   (PAL)
    const unsigned char* In = idr + ((t + 1) & 3) * PL + s;                         // phase ids of layer k+1 (PAL)
    // moduli of the own cell and of its -x / -y neighbours: from the fp64 planes, or through the palette (pal[id] = K,
    // pal[256 + id] = G)
    auto Gof = [&](const double* A, const unsigned char* I, int dx, int dy) -> double {
        return PAL ? pal[256 + I[dy * TX + dx]] : A[3 * PL + dy * TX + dx];
    };
    double* X = sm + Cfg::XCH + PAR * (X_COUNT * PL) + s;                           // this step's exchange planes

    // batch t+1 (layer k+1, set k+1) has landed: it was waited for behind the barrier of the previous step

    // ================= stage A: new stresses =================
    const double vxc = Ac[0 * PL], vyc = Ac[1 * PL], vzc = Ac[2 * PL], Gc = Gof(Ac, Ic, 0, 0);
    const double vxn = An[0 * PL], vyn = An[1 * PL], vzn = An[2 * PL], Gn = Gof(An, In, 0, 0);
    const double Kc = PAL ? pal[Ic[0]] : Bs[0];
    // FORM 1: the old w must be read HERE: after the barrier below the ring-B slot is handed back to the TMA unit
    const double wxo = FORM ? Bs[(BK + 0) * PL] : 0.0, wyo = FORM ? Bs[(BK + 1) * PL] : 0.0, wzo = FORM ? Bs[(BK + 2) * PL] : 0.0;
    const bool bk1 = (k + 1 == 0 || k + 1 == nz);
    const double dxx = (Ac[0 * PL + 1] - vxc) * ih;
    const double dyy = (Ac[1 * PL + TX] - vyc) * ih;
    const double dzz = (vzn - vzc) * ih;
    const double lam_div = fma(-(2.0 / 3.0), Gc, Kc) * (dxx + dyy + dzz);
    const double g2 = 2.0 * Gc;
    // FORM 0: relaxation toward Hooke's law (Eq. 12-13); FORM 1 (displacement form): Hooke's law itself
    const double nsxx = FORM ? fma(g2, dxx, lam_div) : (Bs[(BK + 0) * PL] + th * fma(g2, dxx, lam_div)) * ri;
    const double nsyy = FORM ? fma(g2, dyy, lam_div) : (Bs[(BK + 1) * PL] + th * fma(g2, dyy, lam_div)) * ri;
    const double nszz = FORM ? fma(g2, dzz, lam_div) : (Bs[(BK + 2) * PL] + th * fma(g2, dzz, lam_div)) * ri;
    const double hc = fma(4.0 / 3.0, Gc, Kc);
    const double gl = Gof(Ac, Ic, -1, 0), gd = Gof(Ac, Ic, 0, -1), gld = Gof(Ac, Ic, -1, -1);
    const double gln = Gof(An, In, -1, 0), gdn = Gof(An, In, 0, -1);
    const double gxy = dr_edge_mean_fast<GAVG>(gld, gd, gl, Gc);
    const double gxz = dr_edge_mean_fast<GAVG>(gl, Gc, gln, Gn);
    const double gyz = dr_edge_mean_fast<GAVG>(gd, Gc, gdn, Gn);
    const double vx_d = Ac[0 * PL - TX], vy_l = Ac[1 * PL - 1], vzn_l = An[2 * PL - 1], vzn_d = An[2 * PL - TX];
    double exy = (vxc - vx_d) + (vyc - vy_l);
    double exz = (vxn - vxc) + (vzn - vzn_l);
    double eyz = (vyn - vyc) + (vzn - vzn_d);
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
    const double ntxy = zxy ? 0.0 : (FORM ? gxy * (exy * ih) : (Bs[(BK + 3) * PL] + th * gxy * (exy * ih)) * ri);
    const double ntxz = zxz ? 0.0 : (FORM ? gxz * (exz * ih) : (Bs[(BK + 4) * PL] + th * gxz * (exz * ih)) * ri);
    const double ntyz = zyz ? 0.0 : (FORM ? gyz * (eyz * ih) : (Bs[(BK + 5) * PL] + th * gyz * (eyz * ih)) * ri);

    X[X_SXX * PL] = nsxx; X[X_SYY * PL] = nsyy; X[X_TXY * PL] = ntxy; X[X_HC * PL] = hc; X[X_GXY * PL] = gxy;
    X[X_TXZ * PL] = ntxz; X[X_TYZ * PL] = ntyz; X[X_GXZ * PL] = gxz; X[X_GYZ * PL] = gyz;
    fn.txz = ntxz; fn.tyz = ntyz; fn.gxz = gxz; fn.gyz = gyz; fn.szz = nszz; fn.hc = hc;
    __syncthreads();

    // ---- every thread is done with layer k and set k+1: refill their slots with batch t+4, two steps ahead of need
    if (producer && k + 4 <= ke) {
        const int b = t + 4, m = k + 4;
        unsigned long long* bar = bars + (b & 3);
        double* da = sm + Cfg::RING_A + (b & 3) * (Cfg::NA * PL);
        double* db = sm + Cfg::RING_B + ((b - 1) % 3) * (Cfg::NB * PL);
        dr_tma_issue_batch<FORM, PAL, TX, TY>(T, bar, da, db, idr + (b & 3) * PL, idsrc, idstride, x0, y0, m, true);
    }
    // ---- wait HERE for the batch of the next step (issued two steps ago), not at the top of the next step: stage B
    // below and stage A of the next step then form one straight-line region that the scheduler can interleave
    if (k + 2 <= ke) dr_mbar_wait(bars + ((t + 2) & 3), ((t + 2) >> 2) & 1);

    // ================= stage B: new velocities, stores =================
    if (midrow) {
        const double* Xc = X;      // const view of this step's planes
        // +x / +y neighbours' values on face k+1, carried to the next step (where that face is "face k")
        fn.txz_r = Xc[X_TXZ * PL + 1]; fn.tyz_u = Xc[X_TYZ * PL + TX];
        fn.gxz_r = Xc[X_GXZ * PL + 1]; fn.gyz_u = Xc[X_GYZ * PL + TX];
        if (inner && store) {
            const long long o = sz * k;
            const bool ck = k < nz;                 // k >= 0 here because store implies k >= kb >= 0
            const bool ci = !BND || i < nx, cj = !BND || j < ny;
            if (ck) {
                double nvx = vxc, nvy = vyc;
                double nwx = wxo, nwy = wyo;                 // FORM 1: old w (kept at wall / dead nodes)
                if (cj) {                           // v_x at (i, j+1/2, k+1/2)
                    if (!BND || (i >= 1 && i <= nx - 1)) {
                        const double Fx = ((nsxx - Xc[X_SXX * PL - 1]) + (Xc[X_TXY * PL + TX] - ntxy) + (ntxz - fc.txz)) * ih;
                        const double Hn = dr_max(dr_max(dr_max(Xc[X_HC * PL - 1], hc), dr_max(gxy, Xc[X_GXY * PL + TX])), dr_max(fc.gxz, gxz));
                        if (Hn > 0.0) {
                            const double rH = dr_rcp(Hn);
                            if (RES) { const double r = fabs(Fx) * rH; rnan |= !(r == r); rmax = dr_max(rmax, r); }
                            if (FORM) { nwx = fma(c2t * th * rH, Fx, (1.0 - th) * nwx); nvx = vxc + nwx; }
                            else nvx = fma(c2t * rH, Fx, vxc);
                        }
                    }
                    g.o_vx[o] = nvx;
                    if (FORM) g.o_sxx[o] = nwx; else g.o_txz[o] = fc.txz;
                }
                if (ci) {                           // v_y at (i+1/2, j, k+1/2)
                    if (!BND || (j >= 1 && j <= ny - 1)) {
                        const double Fy = ((Xc[X_TXY * PL + 1] - ntxy) + (nsyy - Xc[X_SYY * PL - TX]) + (ntyz - fc.tyz)) * ih;
                        const double Hn = dr_max(dr_max(dr_max(Xc[X_HC * PL - TX], hc), dr_max(gxy, Xc[X_GXY * PL + 1])), dr_max(fc.gyz, gyz));
                        if (Hn > 0.0) {
                            const double rH = dr_rcp(Hn);
                            if (RES) { const double r = fabs(Fy) * rH; rnan |= !(r == r); rmax = dr_max(rmax, r); }
                            if (FORM) { nwy = fma(c2t * th * rH, Fy, (1.0 - th) * nwy); nvy = vyc + nwy; }
                            else nvy = fma(c2t * rH, Fy, vyc);
                        }
                    }
                    g.o_vy[o] = nvy;
                    if (FORM) g.o_syy[o] = nwy; else g.o_tyz[o] = fc.tyz;
                }
                if (!FORM) {
                    g.o_txy[o] = ntxy;
                    if (ci && cj) { g.o_sxx[o] = nsxx; g.o_syy[o] = nsyy; g.o_szz[o] = nszz; }
                }
            } else if (!FORM) {                     // k == nz: only the top faces
                if (cj) g.o_txz[o] = fc.txz;
                if (ci) g.o_tyz[o] = fc.tyz;
            }
            if (ci && cj) {                         // v_z at (i+1/2, j+1/2, k)
                double nvz = vzc;
                double nwz = wzo;
                if (k >= 1 && k <= nz - 1) {
                    const double Fz = ((fc.txz_r - fc.txz) + (fc.tyz_u - fc.tyz) + (nszz - fc.szz)) * ih;
                    const double Hn = dr_max(dr_max(dr_max(fc.hc, hc), dr_max(fc.gxz, fc.gxz_r)), dr_max(fc.gyz, fc.gyz_u));
                    if (Hn > 0.0) {
                        const double rH = dr_rcp(Hn);
                        if (RES) { const double r = fabs(Fz) * rH; rnan |= !(r == r); rmax = dr_max(rmax, r); }
                        if (FORM) { nwz = fma(c2t * th * rH, Fz, (1.0 - th) * nwz); nvz = vzc + nwz; }
                        else nvz = fma(c2t * rH, Fz, vzc);
                    }
                }
                g.o_vz[o] = nvz;
                if (FORM) g.o_szz[o] = nwz;
            }
        }
    }
}

template <int GAVG, int RES, int FORM, int PAL, int TX, int TY, bool BND>
__device__ __forceinline__ void dr_tma_march(const DrLayout& L, const DrPT& P, const DrTmaps& T, const DrFusedPtrs& g,
                                             double* sm, unsigned char* idr, const double* pal, const unsigned char* idsrc,
                                             const long long idstride, unsigned long long* bars, const int s, const int kb, const int ke,
                                             const int i, const int j, const int x0, const int y0,
                                             const bool producer, const bool midrow, const bool inner, double& rmax, bool& rnan) {
    DrCarry fa, fb;
    fa.txz = fa.tyz = fa.gxz = fa.gyz = fa.szz = fa.hc = fa.txz_r = fa.tyz_u = fa.gxz_r = fa.gyz_u = 0.0;
    fb = fa;
    int k = kb - 1;
    for (int t = 0; k < ke; t += 2, k += 2) {
        dr_tma_step<GAVG, RES, FORM, PAL, TX, TY, BND, 0>(L, P, T, g, sm, idr, pal, idsrc, idstride, bars, s, t, k, kb, ke, k >= kb, i, j, x0, y0, producer, midrow, inner, fa, fb, rmax, rnan);
        if (k + 1 < ke)
            dr_tma_step<GAVG, RES, FORM, PAL, TX, TY, BND, 1>(L, P, T, g, sm, idr, pal, idsrc, idstride, bars, s, t + 1, k + 1, kb, ke, true, i, j, x0, y0, producer, midrow, inner, fb, fa, rmax, rnan);
    }
}

template <int GAVG, int RES, int FORM, int PAL, int TX, int TY>
__global__ void __launch_bounds__(TX * TY, 1)
k_pt_tma(const __grid_constant__ DrTmaps T, DrLayout L, DrPT P, DrFields B, int lz, unsigned long long* res_bits) {
    extern __shared__ __align__(1024) double sm[];
    __shared__ __align__(8) unsigned long long bars[4];
    __shared__ __align__(128) unsigned char idr_raw[PAL ? 128 + 4 * TX * TY + 128 : 16];          // id ring + slack for -1 row reads
    __shared__ double pal[PAL ? 512 : 1];                                                          // K[256], G[256]
    unsigned char* idr = idr_raw + (PAL ? 128 : 0);
    using Cfg = DrTmaCfg2<TX, TY, PAL>;
    constexpr int PL = Cfg::PL;
    const int nx = L.nx, ny = L.ny, nz = L.nz;
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int i0 = blockIdx.x * (TX - 2), j0 = blockIdx.y * (TY - 2);
    const int i = i0 - 1 + tx, j = j0 - 1 + ty;
    const int kb = blockIdx.z * lz;                          // first output layer of this chunk
    const int ke = min(kb + lz, nz + 1);                     // one past the last output layer (layer nz = top faces)
    const int x0 = DR_OX + i0 - 1, y0 = j0;                  // box origin in padded-field coordinates (z = layer + 1)
    const long long idstride = (long long)T.gx * T.gy * (TX * TY);                                   // bytes per layer of ids
    const unsigned char* idsrc = T.ids + ((long long)blockIdx.y * T.gx + blockIdx.x) * (TX * TY);   // this tile, layer -1
    const int s = ty * TX + tx;
    if (PAL) for (int e = s; e < 512; e += TX * TY) pal[e] = T.pal[e];
    const bool producer = (tx == 0 && ty == 0);
    const bool midrow = ty >= 1 && ty <= TY - 2;
    const bool inner = tx >= 1 && tx <= TX - 2 && i <= nx && j <= ny;

    if (producer) {
#pragma unroll
        for (int b = 0; b < 4; ++b) dr_mbar_init(bars + b, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        // prologue: batch 0 = layer kb-1 (ring A only), batches 1..3 = layers kb..kb+2 with their B sets
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const int m = kb - 1 + b;
            if (m <= ke) {
                unsigned long long* bar = bars + b;
                double* da = sm + Cfg::RING_A + b * (Cfg::NA * PL);
                double* db = sm + Cfg::RING_B + (b >= 1 ? b - 1 : 0) * (Cfg::NB * PL);
                dr_tma_issue_batch<FORM, PAL, TX, TY>(T, bar, da, db, idr + b * PL, idsrc, idstride, x0, y0, m, b >= 1);
            }
        }
    }
    __syncthreads();                                          // barrier init visible to every waiter
    dr_mbar_wait(bars + 0, 0);                                // layer kb-1
    dr_mbar_wait(bars + 1, 0);                                // layer kb and set kb (first step)

    const long long qcol = L.origin + min(i, nx + 1) + L.sy * min(j, ny + 1);
    DrFusedPtrs g;
    g.o_vx = B.f[F_VX] + qcol; g.o_vy = B.f[F_VY] + qcol; g.o_vz = B.f[F_VZ] + qcol;
    g.o_sxx = B.f[F_SXX] + qcol; g.o_syy = B.f[F_SYY] + qcol; g.o_szz = B.f[F_SZZ] + qcol;
    g.o_tyz = B.f[F_TYZ] + qcol; g.o_txz = B.f[F_TXZ] + qcol; g.o_txy = B.f[F_TXY] + qcol;
    double rmax = 0.0;
    bool rnan = false;
    const bool interior = i0 >= 2 && i0 + TX - 2 <= nx - 1 && j0 >= 2 && j0 + TY - 2 <= ny - 1;
    if (interior) dr_tma_march<GAVG, RES, FORM, PAL, TX, TY, false>(L, P, T, g, sm, idr, pal, idsrc, idstride, bars, s, kb, ke, i, j, x0, y0, producer, midrow, inner, rmax, rnan);
    else          dr_tma_march<GAVG, RES, FORM, PAL, TX, TY, true>(L, P, T, g, sm, idr, pal, idsrc, idstride, bars, s, kb, ke, i, j, x0, y0, producer, midrow, inner, rmax, rnan);

    if (RES) {
        __shared__ unsigned long long smr[32];
        unsigned long long b = rnan ? 0x7ff8000000000000ull : (unsigned long long)__double_as_longlong(rmax * P.res_scale);
        __syncthreads();
        b = dr_block_max_bits(b, smr);
        if (tx == 0 && ty == 0 && b != 0ull) atomicMax(res_bits, b);
    }
}
