/*
 * dro.cpp -- CPU ORACLE for the pseudo-transient (PT) elasticity iteration of
 * arXiv 2410.20441 (Alkhimenkov, "Digital rock physics: calculation of effective
 * elastic properties of heterogeneous materials using GPUs").
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code
 * with the CUDA path (paper_2410_20441_b200/csrc) and neither includes the other.
 *
 * It is deliberately plain: fp64, straightforward triple loops over the staggered grid,
 * separate p and tau arrays as in the paper (Eq. 10), edge moduli tabulated once per solve,
 * no tiling, no fusion, no reordering.  The only concession to run time is an OpenMP
 * pragma on outer z loops (each loop body writes a distinct node, so results do not
 * depend on the thread count; the max-residual reduction is order independent).
 *
 * Citations: P:NNN = /root/reference/PAPER.md line NNN.  "Reading Rn" = the numbered
 * readings in DESIGN.md (the paper is silent or garbled there).
 *
 * Pins (tests/test_oracle_*.py): homogeneous block = Hooke matrix; affine field is a fixed
 * point; Backus layered medium = Table 2 analytic column; cubic symmetry of a
 * centred sphere; dilute Eshelby pore; Hashin-Shtrikman; Betti symmetry; Eq. 27-29
 * identity; axis permutation; independence of PT constants; dense linear solve of the
 * same discrete problem assembled independently in numpy (brute force, n <= 6); the survey's
 * independent probe numbers incl. iteration counts -- these also
 * cover mean4(gavg=1), the DRO_FORM=1 iterate and, with the zero-by-hand test, apply_void_clamp.
 * Not pinned: closeness to the paper's own *numerical* column of Table 2 (C33 30.419, C44/C55 15.307,
 * C66 25.376, C12 3.720, C13 2.148) and Table 4 (spheroid): geometry garbled at P:194 and
 * shear-test BCs garbled at P:369 -- "parity unpinned" for readings R4/R5 against the paper's own code
 * beyond sign and size of their effect.  A bounded experiment showed that none of
 * the documented readings (gavg 0/1 x bc_mode 0/1) reproduces that column to its printed decimals.
 *
 * DRO_FORM = 1 selects the displacement form of the same discrete problem (state u, w; stresses = Hooke's law of u;
 * w <- (1-theta) w + C~^2 h^2 F/H_node, u <- u + w): not in the paper's text (it cites the method family at P:78), kept
 * because it has the same fixed point -- pinned by tests P10, P10b -- and is the oracle of libdr's DR_FORM = 1.
 *
 * Grid (sec. 3.3, Fig. 1): nx*ny*nz cells of size h, x fastest.
 *   cells  (nx,ny,nz)      : p, txx, tyy, tzz, K, G     at ((i+.5)h,(j+.5)h,(k+.5)h)
 *   vx     (nx+1,ny,nz)    at (i h,(j+.5)h,(k+.5)h);  vy (nx,ny+1,nz);  vz (nx,ny,nz+1)
 *   txy    (nx+1,ny+1,nz)  at (i h, j h,(k+.5)h)
 *   txz    (nx+1,ny,nz+1)  at (i h,(j+.5)h, k h)
 *   tyz    (nx,ny+1,nz+1)  at ((i+.5)h, j h, k h)
 * Voigt order xx,yy,zz,yz,xz,xy ("C55 (xz)" P:365); engineering shear strain.
 * Physical step Delta t = 1, so the paper's velocity is numerically the displacement.
 */
#include <cmath>
#include <cstdio>
#include <cstring>
#include <cstddef>
#include <vector>
#include <string>
#include <algorithm>
#include <chrono>

extern "C" {

enum { DRO_OK = 0, DRO_ERR_ARG = 1, DRO_ERR_WORKSPACE = 2, DRO_ERR_CUDA = 3,
       DRO_ERR_DIVERGED = 4, DRO_ERR_STATE = 5, DRO_MAXITER = 6 };
enum { DRO_CFL = 0, DRO_ST_FACTOR = 1, DRO_NCHECK = 2, DRO_GAVG = 3,
       DRO_VOID_REL = 4, DRO_BC_MODE = 5, DRO_FORM = 8, DRO_STAG_TOL = 10 };
enum { DRO_STOP_NONE = 0, DRO_STOP_RESIDUAL = 1, DRO_STOP_STAGNATION = 2, DRO_STOP_MAXITER = 3 };

struct dro_handle {
    int nx, ny, nz;
    double h;
    std::vector<double> K0, G0;      /* as given                                   */
    std::vector<double> K, G;        /* after the optional void clamp              */
    /* parameters */
    double cfl, st_factor, void_rel;
    double stag_tol;                 /* second stopping rule (reading R9b); 0 = off */
    int stop_reason;                 /* DRO_STOP_* of the last dro_solve */
    int ncheck, gavg, bc_mode;
    int form;                        /* 0 stress-relaxation form of the paper (Eq. 11-13); 1 displacement form */
    /* state */
    std::vector<double> p, txx, tyy, tzz, txy, txz, tyz, vx, vy, vz;
    std::vector<double> wx, wy, wz;  /* displacement form only: damped increments (pseudo-velocities) */
    /* edge shear moduli (O2), tabulated once per solve from K,G by Ctx::Gxy/Gxz/Gyz */
    std::vector<double> eGxy, eGxz, eGyz;
    /* results */
    double Ccol[7][6];               /* Ccol[lc][m] = C[m, lc]; row 6 = <sigma>/eps0 of the triaxial test (App. A.3) */
    bool have[7];
    double avg[6];
    bool have_avg;
    int iters;
    double residual, ms;
    std::string err;
};

} /* extern "C" */

namespace {

struct Grid {
    int nx, ny, nz;
    inline size_t c(int i, int j, int k) const { return (size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * k); }
    inline size_t fx(int i, int j, int k) const { return (size_t)i + (size_t)(nx + 1) * ((size_t)j + (size_t)ny * k); }
    inline size_t fy(int i, int j, int k) const { return (size_t)i + (size_t)nx * ((size_t)j + (size_t)(ny + 1) * k); }
    inline size_t fz(int i, int j, int k) const { return (size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * k); }
    inline size_t exy(int i, int j, int k) const { return (size_t)i + (size_t)(nx + 1) * ((size_t)j + (size_t)(ny + 1) * k); }
    inline size_t exz(int i, int j, int k) const { return (size_t)i + (size_t)(nx + 1) * ((size_t)j + (size_t)ny * k); }
    inline size_t eyz(int i, int j, int k) const { return (size_t)i + (size_t)nx * ((size_t)j + (size_t)(ny + 1) * k); }
};

inline int clampi(int a, int lo, int hi) { return a < lo ? lo : (a > hi ? hi : a); }

/* Reading R4 (paper silent; BASELINE "moduli averaged onto shear nodes"): the shear modulus on
 * an edge is the harmonic mean of the four cells round it, 0 if any of them is 0; cells missing
 * outside the domain are replaced by their mirror image (replicate padding).  gavg=1: arithmetic. */
inline double mean4(double a, double b, double c, double d, int gavg) {
    if (gavg == 1) return 0.25 * (a + b + c + d);
    if (a == 0.0 || b == 0.0 || c == 0.0 || d == 0.0) return 0.0;
    return 4.0 / (1.0 / a + 1.0 / b + 1.0 / c + 1.0 / d);
}

struct Ctx {
    const dro_handle* H;
    Grid g;
    const double* G;
    const double* K;
    int gavg;
    /* cell shear modulus with replicate padding */
    inline double Gc(int i, int j, int k) const {
        return G[g.c(clampi(i, 0, g.nx - 1), clampi(j, 0, g.ny - 1), clampi(k, 0, g.nz - 1))];
    }
    inline double Hc(int i, int j, int k) const {       /* P-wave modulus K + 4G/3 */
        size_t q = g.c(i, j, k);
        return K[q] + 4.0 * G[q] / 3.0;
    }
    /* edge moduli; edge (i,j,k) of family xy sits at (i h, j h, (k+.5) h) etc. */
    inline double Gxy(int i, int j, int k) const { return mean4(Gc(i - 1, j - 1, k), Gc(i, j - 1, k), Gc(i - 1, j, k), Gc(i, j, k), gavg); }
    inline double Gxz(int i, int j, int k) const { return mean4(Gc(i - 1, j, k - 1), Gc(i, j, k - 1), Gc(i - 1, j, k), Gc(i, j, k), gavg); }
    inline double Gyz(int i, int j, int k) const { return mean4(Gc(i, j - 1, k - 1), Gc(i, j, k - 1), Gc(i, j - 1, k), Gc(i, j, k), gavg); }
};

/* Load case -> displacement gradient D (reading R6; P:347-357 A.1, P:365-369 A.2):
 * lc 0,1,2: Dxx,Dyy,Dzz = eps0;  lc 3 (yz): u_y = eps0 z;  lc 4 (xz): u_x = eps0 z;  lc 5 (xy): u_x = eps0 y.
 * lc 6: the 7th direct test of App. A.3: the normal displacement of all three face pairs is prescribed at
 * once (Dxx = Dyy = Dzz = eps0), tangential components free as in the normal tests. */
struct Affine {
    double D[3][3];
    Affine(int lc, double e) {
        for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) D[a][b] = 0.0;
        switch (lc) {
            case 0: D[0][0] = e; break;
            case 1: D[1][1] = e; break;
            case 2: D[2][2] = e; break;
            case 3: D[1][2] = e; break;
            case 4: D[0][2] = e; break;
            case 5: D[0][1] = e; break;
            case 6: D[0][0] = e; D[1][1] = e; D[2][2] = e; break;
        }
    }
    inline double u(int a, double x, double y, double z) const { return D[a][0] * x + D[a][1] * y + D[a][2] * z; }
};

/* is shear component (Voigt 3=yz, 4=xz, 5=xy) computed on boundary edges (ghost rule) or zero?
 * Reading R5 (P:371 cannot hold a uniform simple shear; P:369 garbled): only the loaded plane of
 * lc 3-5 is prescribed on the faces; bc_mode=1 prescribes all (full kinematic uniform BC). */
inline bool ghost_on(int voigt, int lc, int bc_mode) { return bc_mode == 1 || voigt == lc; }

void apply_void_clamp(dro_handle* H) {
    H->K = H->K0; H->G = H->G0;
    if (H->void_rel > 0.0) {
        double hmax = 0.0;
        for (size_t q = 0; q < H->K.size(); ++q) hmax = std::max(hmax, H->K[q] + 4.0 * H->G[q] / 3.0);
        for (size_t q = 0; q < H->K.size(); ++q)
            if (H->K[q] + 4.0 * H->G[q] / 3.0 <= H->void_rel * hmax) { H->K[q] = 0.0; H->G[q] = 0.0; }
    }
}

/* O5 initial fields (reading R8): every velocity node := affine u0 at its own position;
 * stresses := local Hooke's law of the uniform strain E = sym(D). */
void init_fields(dro_handle* H, int lc, double eps0) {
    apply_void_clamp(H);
    const int nx = H->nx, ny = H->ny, nz = H->nz;
    const double h = H->h;
    Grid g{nx, ny, nz};
    Ctx cx{H, g, H->G.data(), H->K.data(), H->gavg};
    Affine A(lc, eps0);
    const double Exx = A.D[0][0], Eyy = A.D[1][1], Ezz = A.D[2][2];
    const double gyz = A.D[1][2] + A.D[2][1], gxz = A.D[0][2] + A.D[2][0], gxy = A.D[0][1] + A.D[1][0];
    const double trE = Exx + Eyy + Ezz;
    const size_t N = (size_t)nx * ny * nz;
    H->p.assign(N, 0.0); H->txx.assign(N, 0.0); H->tyy.assign(N, 0.0); H->tzz.assign(N, 0.0);
    H->vx.assign((size_t)(nx + 1) * ny * nz, 0.0);
    H->vy.assign((size_t)nx * (ny + 1) * nz, 0.0);
    H->vz.assign((size_t)nx * ny * (nz + 1), 0.0);
    H->wx.assign(H->vx.size(), 0.0); H->wy.assign(H->vy.size(), 0.0); H->wz.assign(H->vz.size(), 0.0);
    H->txy.assign((size_t)(nx + 1) * (ny + 1) * nz, 0.0);
    H->txz.assign((size_t)(nx + 1) * ny * (nz + 1), 0.0);
    H->tyz.assign((size_t)nx * (ny + 1) * (nz + 1), 0.0);
    H->eGxy.assign(H->txy.size(), 0.0); H->eGxz.assign(H->txz.size(), 0.0); H->eGyz.assign(H->tyz.size(), 0.0);
    for (int k = 0; k < nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i <= nx; ++i) H->eGxy[g.exy(i, j, k)] = cx.Gxy(i, j, k);
    for (int k = 0; k <= nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i <= nx; ++i) H->eGxz[g.exz(i, j, k)] = cx.Gxz(i, j, k);
    for (int k = 0; k <= nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i < nx; ++i) H->eGyz[g.eyz(i, j, k)] = cx.Gyz(i, j, k);
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i <= nx; ++i)
        H->vx[g.fx(i, j, k)] = A.u(0, i * h, (j + 0.5) * h, (k + 0.5) * h);
    for (int k = 0; k < nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i < nx; ++i)
        H->vy[g.fy(i, j, k)] = A.u(1, (i + 0.5) * h, j * h, (k + 0.5) * h);
    for (int k = 0; k <= nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i)
        H->vz[g.fz(i, j, k)] = A.u(2, (i + 0.5) * h, (j + 0.5) * h, k * h);
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
        size_t q = g.c(i, j, k);
        H->p[q] = -H->K[q] * trE;
        H->txx[q] = 2.0 * H->G[q] * (Exx - trE / 3.0);
        H->tyy[q] = 2.0 * H->G[q] * (Eyy - trE / 3.0);
        H->tzz[q] = 2.0 * H->G[q] * (Ezz - trE / 3.0);
    }
    for (int k = 0; k < nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i <= nx; ++i) {
        bool bnd = (i == 0 || i == nx || j == 0 || j == ny);
        H->txy[g.exy(i, j, k)] = (bnd && !ghost_on(5, lc, H->bc_mode)) ? 0.0 : H->eGxy[g.exy(i, j, k)] * gxy;
    }
    for (int k = 0; k <= nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i <= nx; ++i) {
        bool bnd = (i == 0 || i == nx || k == 0 || k == nz);
        H->txz[g.exz(i, j, k)] = (bnd && !ghost_on(4, lc, H->bc_mode)) ? 0.0 : H->eGxz[g.exz(i, j, k)] * gxz;
    }
    for (int k = 0; k <= nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i < nx; ++i) {
        bool bnd = (j == 0 || j == ny || k == 0 || k == nz);
        H->tyz[g.eyz(i, j, k)] = (bnd && !ghost_on(3, lc, H->bc_mode)) ? 0.0 : H->eGyz[g.eyz(i, j, k)] * gyz;
    }
}

/* O7: one PT iteration.  Returns the residual of this iteration's velocity update
 * (max over updated nodes of |F| h / (H_node |eps0|)) when want_res, else 0. */
double pt_iteration(dro_handle* H, int lc, double eps0, bool want_res) {
    const int nx = H->nx, ny = H->ny, nz = H->nz;
    const double h = H->h;
    Grid g{nx, ny, nz};
    Ctx cx{H, g, H->G.data(), H->K.data(), H->gavg};
    Affine A(lc, eps0);
    const double Lx = nx * h, Ly = ny * h, Lz = nz * h;
    /* O1 (Eq. 14, 16 P:98-107; St_opt = 2 pi sqrt(3) in 3-D): theta = dt~/Dt =
     * C~ St h / L_max with local numerical moduli K~ = K(x), G~ = G(x) (reading R2). */
    const int nmax = std::max(nx, std::max(ny, nz));
    const double St = 2.0 * M_PI * std::sqrt(3.0) * H->st_factor;
    const double theta = H->cfl * St / nmax;
    /* Eq. 17 P:111 with L/(St Dt) = C~ h / theta:  dt~/rho~ = C~^2 h^2 / (theta H_node) */
    const double c2 = H->cfl * H->cfl * h * h;
    double *p = H->p.data(), *txx = H->txx.data(), *tyy = H->tyy.data(), *tzz = H->tzz.data();
    double *txy = H->txy.data(), *txz = H->txz.data(), *tyz = H->tyz.data();
    double *vx = H->vx.data(), *vy = H->vy.data(), *vz = H->vz.data();
    const double* K = H->K.data();
    const double* G = H->G.data();
    const int bcm = H->bc_mode;
    const int form = H->form;
    double *wx = H->wx.data(), *wy = H->wy.data(), *wz = H->wz.data();
    const double *eGxy = H->eGxy.data(), *eGxz = H->eGxz.data(), *eGyz = H->eGyz.data();

    /* ---- 1. stress update (Eq. 12-13, relaxation term implicit: reading R14) ---- */
    #pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
        size_t q = g.c(i, j, k);
        double dxx = (vx[g.fx(i + 1, j, k)] - vx[g.fx(i, j, k)]) / h;
        double dyy = (vy[g.fy(i, j + 1, k)] - vy[g.fy(i, j, k)]) / h;
        double dzz = (vz[g.fz(i, j, k + 1)] - vz[g.fz(i, j, k)]) / h;
        double div = dxx + dyy + dzz;
        if (form == 0) {
        p[q] = (p[q] - theta * K[q] * div) / (1.0 + theta);
        txx[q] = (txx[q] + theta * 2.0 * G[q] * (dxx - div / 3.0)) / (1.0 + theta);
        tyy[q] = (tyy[q] + theta * 2.0 * G[q] * (dyy - div / 3.0)) / (1.0 + theta);
        tzz[q] = (tzz[q] + theta * 2.0 * G[q] * (dzz - div / 3.0)) / (1.0 + theta);
        } else {                 /* displacement form: stresses are Hooke's law of the current displacement */
        p[q] = -K[q] * div;
        txx[q] = 2.0 * G[q] * (dxx - div / 3.0);
        tyy[q] = 2.0 * G[q] * (dyy - div / 3.0);
        tzz[q] = 2.0 * G[q] * (dzz - div / 3.0);
        }
    }
    /* shear stresses on edges; boundary edges per O6 rule T (ghost value so that the wall value is affine) */
    #pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i <= nx; ++i) {
        size_t e = g.exy(i, j, k);
        bool bnd = (i == 0 || i == nx || j == 0 || j == ny);
        if (bnd && !ghost_on(5, lc, bcm)) { txy[e] = 0.0; continue; }
        double z = (k + 0.5) * h;
        double dvx_dy, dvy_dx;
        if (j == 0)       dvx_dy = 2.0 * (vx[g.fx(i, 0, k)] - A.u(0, i * h, 0.0, z)) / h;
        else if (j == ny) dvx_dy = 2.0 * (A.u(0, i * h, Ly, z) - vx[g.fx(i, ny - 1, k)]) / h;
        else              dvx_dy = (vx[g.fx(i, j, k)] - vx[g.fx(i, j - 1, k)]) / h;
        if (i == 0)       dvy_dx = 2.0 * (vy[g.fy(0, j, k)] - A.u(1, 0.0, j * h, z)) / h;
        else if (i == nx) dvy_dx = 2.0 * (A.u(1, Lx, j * h, z) - vy[g.fy(nx - 1, j, k)]) / h;
        else              dvy_dx = (vy[g.fy(i, j, k)] - vy[g.fy(i - 1, j, k)]) / h;
        if (form == 0) txy[e] = (txy[e] + theta * eGxy[g.exy(i, j, k)] * (dvx_dy + dvy_dx)) / (1.0 + theta);
        else           txy[e] = eGxy[g.exy(i, j, k)] * (dvx_dy + dvy_dx);
    }
    #pragma omp parallel for schedule(static)
    for (int k = 0; k <= nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i <= nx; ++i) {
        size_t e = g.exz(i, j, k);
        bool bnd = (i == 0 || i == nx || k == 0 || k == nz);
        if (bnd && !ghost_on(4, lc, bcm)) { txz[e] = 0.0; continue; }
        double y = (j + 0.5) * h;
        double dvx_dz, dvz_dx;
        if (k == 0)       dvx_dz = 2.0 * (vx[g.fx(i, j, 0)] - A.u(0, i * h, y, 0.0)) / h;
        else if (k == nz) dvx_dz = 2.0 * (A.u(0, i * h, y, Lz) - vx[g.fx(i, j, nz - 1)]) / h;
        else              dvx_dz = (vx[g.fx(i, j, k)] - vx[g.fx(i, j, k - 1)]) / h;
        if (i == 0)       dvz_dx = 2.0 * (vz[g.fz(0, j, k)] - A.u(2, 0.0, y, k * h)) / h;
        else if (i == nx) dvz_dx = 2.0 * (A.u(2, Lx, y, k * h) - vz[g.fz(nx - 1, j, k)]) / h;
        else              dvz_dx = (vz[g.fz(i, j, k)] - vz[g.fz(i - 1, j, k)]) / h;
        if (form == 0) txz[e] = (txz[e] + theta * eGxz[g.exz(i, j, k)] * (dvx_dz + dvz_dx)) / (1.0 + theta);
        else           txz[e] = eGxz[g.exz(i, j, k)] * (dvx_dz + dvz_dx);
    }
    #pragma omp parallel for schedule(static)
    for (int k = 0; k <= nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i < nx; ++i) {
        size_t e = g.eyz(i, j, k);
        bool bnd = (j == 0 || j == ny || k == 0 || k == nz);
        if (bnd && !ghost_on(3, lc, bcm)) { tyz[e] = 0.0; continue; }
        double x = (i + 0.5) * h;
        double dvy_dz, dvz_dy;
        if (k == 0)       dvy_dz = 2.0 * (vy[g.fy(i, j, 0)] - A.u(1, x, j * h, 0.0)) / h;
        else if (k == nz) dvy_dz = 2.0 * (A.u(1, x, j * h, Lz) - vy[g.fy(i, j, nz - 1)]) / h;
        else              dvy_dz = (vy[g.fy(i, j, k)] - vy[g.fy(i, j, k - 1)]) / h;
        if (j == 0)       dvz_dy = 2.0 * (vz[g.fz(i, 0, k)] - A.u(2, x, 0.0, k * h)) / h;
        else if (j == ny) dvz_dy = 2.0 * (A.u(2, x, Ly, k * h) - vz[g.fz(i, ny - 1, k)]) / h;
        else              dvz_dy = (vz[g.fz(i, j, k)] - vz[g.fz(i, j - 1, k)]) / h;
        if (form == 0) tyz[e] = (tyz[e] + theta * eGyz[g.eyz(i, j, k)] * (dvy_dz + dvz_dy)) / (1.0 + theta);
        else           tyz[e] = eGyz[g.eyz(i, j, k)] * (dvy_dz + dvz_dy);
    }

    /* ---- 2. velocity update with the NEW stresses (Eq. 11); wall nodes untouched (O6 rule N).
     * H_node (reading R3) = stiffest of the six springs in the node's stencil. ---- */
    double res = 0.0;
    const double ae = std::fabs(eps0);
    #pragma omp parallel for schedule(static) reduction(max : res)
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 1; i < nx; ++i) {
        double sxx1 = -p[g.c(i, j, k)] + txx[g.c(i, j, k)];
        double sxx0 = -p[g.c(i - 1, j, k)] + txx[g.c(i - 1, j, k)];
        double F = (sxx1 - sxx0) / h + (txy[g.exy(i, j + 1, k)] - txy[g.exy(i, j, k)]) / h
                 + (txz[g.exz(i, j, k + 1)] - txz[g.exz(i, j, k)]) / h;
        double Hn = std::max(std::max(cx.Hc(i - 1, j, k), cx.Hc(i, j, k)),
                             std::max(std::max(eGxy[g.exy(i, j, k)], eGxy[g.exy(i, j + 1, k)]),
                                      std::max(eGxz[g.exz(i, j, k)], eGxz[g.exz(i, j, k + 1)])));
        if (Hn > 0.0) {
            if (want_res) { double r = std::fabs(F) * h / (Hn * ae); if (!(r <= res)) res = r; }
            if (form == 0) vx[g.fx(i, j, k)] += c2 / (theta * Hn) * F;
            else { size_t n = g.fx(i, j, k); wx[n] = (1.0 - theta) * wx[n] + c2 / Hn * F; vx[n] += wx[n]; }
        }
    }
    #pragma omp parallel for schedule(static) reduction(max : res)
    for (int k = 0; k < nz; ++k) for (int j = 1; j < ny; ++j) for (int i = 0; i < nx; ++i) {
        double syy1 = -p[g.c(i, j, k)] + tyy[g.c(i, j, k)];
        double syy0 = -p[g.c(i, j - 1, k)] + tyy[g.c(i, j - 1, k)];
        double F = (txy[g.exy(i + 1, j, k)] - txy[g.exy(i, j, k)]) / h + (syy1 - syy0) / h
                 + (tyz[g.eyz(i, j, k + 1)] - tyz[g.eyz(i, j, k)]) / h;
        double Hn = std::max(std::max(cx.Hc(i, j - 1, k), cx.Hc(i, j, k)),
                             std::max(std::max(eGxy[g.exy(i, j, k)], eGxy[g.exy(i + 1, j, k)]),
                                      std::max(eGyz[g.eyz(i, j, k)], eGyz[g.eyz(i, j, k + 1)])));
        if (Hn > 0.0) {
            if (want_res) { double r = std::fabs(F) * h / (Hn * ae); if (!(r <= res)) res = r; }
            if (form == 0) vy[g.fy(i, j, k)] += c2 / (theta * Hn) * F;
            else { size_t n = g.fy(i, j, k); wy[n] = (1.0 - theta) * wy[n] + c2 / Hn * F; vy[n] += wy[n]; }
        }
    }
    #pragma omp parallel for schedule(static) reduction(max : res)
    for (int k = 1; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
        double szz1 = -p[g.c(i, j, k)] + tzz[g.c(i, j, k)];
        double szz0 = -p[g.c(i, j, k - 1)] + tzz[g.c(i, j, k - 1)];
        double F = (txz[g.exz(i + 1, j, k)] - txz[g.exz(i, j, k)]) / h
                 + (tyz[g.eyz(i, j + 1, k)] - tyz[g.eyz(i, j, k)]) / h + (szz1 - szz0) / h;
        double Hn = std::max(std::max(cx.Hc(i, j, k - 1), cx.Hc(i, j, k)),
                             std::max(std::max(eGxz[g.exz(i, j, k)], eGxz[g.exz(i + 1, j, k)]),
                                      std::max(eGyz[g.eyz(i, j, k)], eGyz[g.eyz(i, j + 1, k)])));
        if (Hn > 0.0) {
            if (want_res) { double r = std::fabs(F) * h / (Hn * ae); if (!(r <= res)) res = r; }
            if (form == 0) vz[g.fz(i, j, k)] += c2 / (theta * Hn) * F;
            else { size_t n = g.fz(i, j, k); wz[n] = (1.0 - theta) * wz[n] + c2 / Hn * F; vz[n] += wz[n]; }
        }
    }
    return res;
}

/* O8 (Eq. 7; reading R7): cell mean for normal stresses, trapezoid-weighted mean for edge shears.
 * Eq. 7 is an exact sum; the oracle evaluates it to fp64 working precision (reading R7b in DESIGN.md): the same plain
 * sequential loops, with the running sums kept in long double (x87 extended, 64-bit mantissa).  A double accumulator over
 * the 1.1e8 terms of a 479^3 image carried 5e-11 of rounding -- within 2x of the 1e-10 the stagnation rule R9b decides on,
 * and more than the kernel's pairwise sum (1e-15); with long double the sum is good to ~1e-15 and rounded once at the end. */
void volume_averages(const dro_handle* H, double out[6]) {
    const int nx = H->nx, ny = H->ny, nz = H->nz;
    Grid g{nx, ny, nz};
    const long double N = (long double)nx * ny * nz;
    long double s[6] = {0, 0, 0, 0, 0, 0};
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
        size_t q = g.c(i, j, k);
        s[0] += -H->p[q] + H->txx[q];
        s[1] += -H->p[q] + H->tyy[q];
        s[2] += -H->p[q] + H->tzz[q];
    }
    auto w = [](int a, int n) { return (a == 0 || a == n) ? 0.5 : 1.0; };
    for (int k = 0; k <= nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i < nx; ++i)
        s[3] += w(j, ny) * w(k, nz) * H->tyz[g.eyz(i, j, k)];
    for (int k = 0; k <= nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i <= nx; ++i)
        s[4] += w(i, nx) * w(k, nz) * H->txz[g.exz(i, j, k)];
    for (int k = 0; k < nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i <= nx; ++i)
        s[5] += w(i, nx) * w(j, ny) * H->txy[g.exy(i, j, k)];
    for (int m = 0; m < 6; ++m) out[m] = (double)(s[m] / N);
}

void store_column(dro_handle* H, int lc, double eps0) {
    volume_averages(H, H->avg);
    H->have_avg = true;
    for (int m = 0; m < 6; ++m) H->Ccol[lc][m] = H->avg[m] / eps0;   /* Eq. 9, 22 P:70 */
    H->have[lc] = true;
}

bool bad_solve_args(dro_handle* H, int lc, double eps0) {
    if (!H) return true;
    if (lc < 0 || lc > 6 || !(eps0 != 0.0) || !std::isfinite(eps0)) { H->err = "bad load case or eps0"; return true; }
    return false;
}

} /* namespace */

extern "C" {

int dro_create(int nx, int ny, int nz, double h, const double* K, const double* G, dro_handle** out) {
    if (!out) return DRO_ERR_ARG;
    *out = nullptr;
    if (nx < 2 || ny < 2 || nz < 2 || !(h > 0.0) || !K || !G) return DRO_ERR_ARG;
    size_t N = (size_t)nx * ny * nz;
    for (size_t q = 0; q < N; ++q)
        if (!(K[q] >= 0.0) || !(G[q] >= 0.0) || !std::isfinite(K[q]) || !std::isfinite(G[q])) return DRO_ERR_ARG;
    dro_handle* H = new dro_handle();
    H->nx = nx; H->ny = ny; H->nz = nz; H->h = h;
    H->K0.assign(K, K + N); H->G0.assign(G, G + N);
    H->cfl = 0.55; H->st_factor = 1.0; H->void_rel = 0.0; H->ncheck = 50; H->gavg = 0; H->bc_mode = 0; H->form = 0;
    H->stag_tol = 1e-10; H->stop_reason = DRO_STOP_NONE;
    for (int a = 0; a < 7; ++a) { H->have[a] = false; for (int b = 0; b < 6; ++b) H->Ccol[a][b] = 0.0; }
    H->have_avg = false; H->iters = 0; H->residual = 0.0; H->ms = 0.0;
    *out = H;
    return DRO_OK;
}

int dro_set_param(dro_handle* H, int id, double value) {
    if (!H) return DRO_ERR_ARG;
    switch (id) {
        case DRO_CFL:       if (!(value > 0.0)) break; H->cfl = value; return DRO_OK;
        case DRO_ST_FACTOR: if (!(value > 0.0)) break; H->st_factor = value; return DRO_OK;
        case DRO_NCHECK:    if (!(value >= 1.0)) break; H->ncheck = (int)value; return DRO_OK;
        case DRO_GAVG:      if (value != 0.0 && value != 1.0) break; H->gavg = (int)value; return DRO_OK;
        case DRO_VOID_REL:  if (!(value >= 0.0)) break; H->void_rel = value; return DRO_OK;
        case DRO_BC_MODE:   if (value != 0.0 && value != 1.0) break; H->bc_mode = (int)value; return DRO_OK;
        /* the explicit damping of the displacement form has a smaller stability margin (diverges at C~ = 0.55 on
           small grids, converges at 0.52): choosing a form also resets C~ to that form's default */
        case DRO_FORM:      if (value != 0.0 && value != 1.0) break; H->form = (int)value; H->cfl = H->form ? 0.50 : 0.55; return DRO_OK;
        case DRO_STAG_TOL:  if (!(value >= 0.0)) break; H->stag_tol = value; return DRO_OK;
        default: break;
    }
    H->err = "bad parameter id or value";
    return DRO_ERR_ARG;
}

/* O7.3: iterate; every ncheck iterations test res <= tol ("once the dynamic fields attenuate to a certain
 * precision").
 * Second rule (reading R9b in DESIGN.md; the paper states no stopping rule beyond P:78): with tiny-but-non-zero pore
 * moduli the max-norm plateaus in the pores (H_node ~ 1e-6 of the matrix) while <sigma>, the only thing Eq. 9/22 use,
 * no longer moves.  So at every check where res > tol the volume averages (O8) are formed and compared with those of
 * the previous comparison: d = max_m |<sigma_m> - <sigma_m>_prev| / max_m |<sigma_m>|.  Two consecutive comparisons with
 * d <= stag_tol (default 1e-10, four orders below the 1e-6 bar on C) stop the solve with DRO_OK and
 * stop_reason = DRO_STOP_STAGNATION.  stag_tol = 0 switches the rule off.
 * The movement is measured over at least DRO_STAG_WINDOW = 50 iterations: a check that comes sooner after the last
 * comparison than that is skipped by this rule (with ncheck = 1 the per-iteration movement would drop below stag_tol long
 * before <sigma> has converged; the error left at the stop is about d rho^w / (1 - rho^w) for a contraction rate rho per
 * iteration and a window of w iterations).  For ncheck >= 50 every check compares, as before. */
#define DRO_STAG_WINDOW 50
int dro_solve(dro_handle* H, int lc, double eps0, double tol, int maxiter) {
    if (bad_solve_args(H, lc, eps0)) return DRO_ERR_ARG;
    if (!(tol > 0.0) || maxiter < 1) { H->err = "bad tol or maxiter"; return DRO_ERR_ARG; }
    auto t0 = std::chrono::steady_clock::now();
    init_fields(H, lc, eps0);
    int status = DRO_MAXITER;
    H->residual = INFINITY;
    H->stop_reason = DRO_STOP_MAXITER;
    bool have_prev = false;
    double prev[6] = {0, 0, 0, 0, 0, 0};
    int calm = 0;
    int prev_it = 0;
    int it = 0;
    for (it = 1; it <= maxiter; ++it) {
        bool chk = (it % H->ncheck == 0);
        double r = pt_iteration(H, lc, eps0, chk);
        if (chk) {
            H->residual = r;
            if (!std::isfinite(r)) { status = DRO_ERR_DIVERGED; H->stop_reason = DRO_STOP_NONE; break; }
            if (r <= tol) { status = DRO_OK; H->stop_reason = DRO_STOP_RESIDUAL; break; }
            if (H->stag_tol > 0.0 && (!have_prev || it - prev_it >= DRO_STAG_WINDOW)) {
                double a[6], num = 0.0, den = 0.0;
                volume_averages(H, a);
                for (int m = 0; m < 6; ++m) { num = std::max(num, std::fabs(a[m] - prev[m])); den = std::max(den, std::fabs(a[m])); }
                if (have_prev && num <= H->stag_tol * den) ++calm; else calm = 0;
                for (int m = 0; m < 6; ++m) prev[m] = a[m];
                have_prev = true; prev_it = it;
                if (calm >= 2) { status = DRO_OK; H->stop_reason = DRO_STOP_STAGNATION; break; }
            }
        }
    }
    H->iters = std::min(it, maxiter);
    H->ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
    if (status == DRO_ERR_DIVERGED) { H->err = "residual is not finite"; return status; }
    store_column(H, lc, eps0);
    return status;
}

int dro_stop_reason(dro_handle* H) { return H ? H->stop_reason : DRO_STOP_NONE; }

/* fixed iteration count (parity): init, niter iterations, residual of the last one, averages. */
int dro_step(dro_handle* H, int lc, double eps0, int niter) {
    if (bad_solve_args(H, lc, eps0)) return DRO_ERR_ARG;
    if (niter < 0) { H->err = "bad niter"; return DRO_ERR_ARG; }
    auto t0 = std::chrono::steady_clock::now();
    init_fields(H, lc, eps0);
    double r = 0.0;
    for (int it = 1; it <= niter; ++it) r = pt_iteration(H, lc, eps0, it == niter);
    H->iters = niter; H->residual = r;
    H->ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
    store_column(H, lc, eps0);
    return DRO_OK;
}

/* continue iterating from the current fields (timing of the bare iteration; no init, no averages) */
int dro_iterate(dro_handle* H, int lc, double eps0, int niter) {
    if (bad_solve_args(H, lc, eps0)) return DRO_ERR_ARG;
    if (H->p.empty()) { H->err = "no fields: call dro_step/dro_solve first"; return DRO_ERR_STATE; }
    auto t0 = std::chrono::steady_clock::now();
    for (int it = 1; it <= niter; ++it) pt_iteration(H, lc, eps0, false);
    H->ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
    return DRO_OK;
}

int dro_effective_C(dro_handle* H, double out[36]) {
    if (!H || !out) return DRO_ERR_ARG;
    for (int lc = 0; lc < 6; ++lc) if (!H->have[lc]) { H->err = "not all six load cases solved"; return DRO_ERR_STATE; }
    for (int m = 0; m < 6; ++m) for (int lc = 0; lc < 6; ++lc) out[6 * m + lc] = H->Ccol[lc][m];
    return DRO_OK;
}

/* Eq. 24-29: off-diagonal normal components from the 7th (triaxial) test.  With eps_k = eps0 in all three
 * directions, sigma_bar_k = <sigma_kk> - C_kk eps_k (Eq. 24, C_kk from the direct normal tests lc 0-2) and
 * eps_bar_k = eps_k (Eq. 25):  out = (C12, C13, C23) of Eq. 27, 28, 29.  Ccol[6] holds <sigma>/eps0 of the triaxial test,
 * so eps0 cancels: sb_k = Ccol[6][k] - Ccol[k][k] and eb_k = 1. */
int dro_offdiag_direct(dro_handle* H, double out[3]) {
    if (!H || !out) return DRO_ERR_ARG;
    for (int lc : {0, 1, 2, 6}) if (!H->have[lc]) { H->err = "needs load cases 0, 1, 2 and 6"; return DRO_ERR_STATE; }
    const double sb1 = H->Ccol[6][0] - H->Ccol[0][0], sb2 = H->Ccol[6][1] - H->Ccol[1][1], sb3 = H->Ccol[6][2] - H->Ccol[2][2];
    const double e1 = 1.0, e2 = 1.0, e3 = 1.0;
    out[0] = (e1 * sb1 + e2 * sb2 - e3 * sb3) / (2.0 * e1 * e2);     /* Eq. 27 */
    out[1] = (e1 * sb1 - e2 * sb2 + e3 * sb3) / (2.0 * e1 * e3);     /* Eq. 28 */
    out[2] = (-e1 * sb1 + e2 * sb2 + e3 * sb3) / (2.0 * e2 * e3);    /* Eq. 29 */
    return DRO_OK;
}

int dro_avg_stress(dro_handle* H, double out[6]) {
    if (!H || !out) return DRO_ERR_ARG;
    if (!H->have_avg) { H->err = "no solve yet"; return DRO_ERR_STATE; }
    for (int m = 0; m < 6; ++m) out[m] = H->avg[m];
    return DRO_OK;
}

int dro_info(dro_handle* H, int* iters, double* residual, double* ms) {
    if (!H) return DRO_ERR_ARG;
    if (iters) *iters = H->iters;
    if (residual) *residual = H->residual;
    if (ms) *ms = H->ms;
    return DRO_OK;
}

/* fields 0..8: vx vy vz sxx syy szz tyz txz txy, dense logical shape, x fastest; sigma_aa = -p + tau_aa (Eq. 10) */
size_t dro_field_size(dro_handle* H, int field) {
    if (!H) return 0;
    size_t nx = H->nx, ny = H->ny, nz = H->nz;
    switch (field) {
        case 0: return (nx + 1) * ny * nz;
        case 1: return nx * (ny + 1) * nz;
        case 2: return nx * ny * (nz + 1);
        case 3: case 4: case 5: return nx * ny * nz;
        case 6: return nx * (ny + 1) * (nz + 1);
        case 7: return (nx + 1) * ny * (nz + 1);
        case 8: return (nx + 1) * (ny + 1) * nz;
    }
    return 0;
}

int dro_get_field(dro_handle* H, int field, double* dst, size_t n) {
    if (!H || !dst) return DRO_ERR_ARG;
    size_t need = dro_field_size(H, field);
    if (need == 0 || n != need) { H->err = "bad field id or size"; return DRO_ERR_ARG; }
    if (H->p.empty()) { H->err = "no fields yet"; return DRO_ERR_STATE; }
    const std::vector<double>* src = nullptr;
    switch (field) {
        case 0: src = &H->vx; break; case 1: src = &H->vy; break; case 2: src = &H->vz; break;
        case 6: src = &H->tyz; break; case 7: src = &H->txz; break; case 8: src = &H->txy; break;
        default: break;
    }
    if (src) { std::memcpy(dst, src->data(), need * sizeof(double)); return DRO_OK; }
    const std::vector<double>& t = field == 3 ? H->txx : (field == 4 ? H->tyy : H->tzz);
    for (size_t q = 0; q < need; ++q) dst[q] = -H->p[q] + t[q];
    return DRO_OK;
}

/* raw state arrays for the z-slab halo test (tests/test_shard_gloo.py): 0 vx 1 vy 2 vz 3 p 4 txx 5 tyy 6 tzz 7 tyz 8 txz 9 txy,
 * whole arrays, dense logical shape.  Pure copies: no arithmetic. */
static std::vector<double>* raw_array(dro_handle* H, int id) {
    switch (id) {
        case 0: return &H->vx; case 1: return &H->vy; case 2: return &H->vz; case 3: return &H->p; case 4: return &H->txx;
        case 5: return &H->tyy; case 6: return &H->tzz; case 7: return &H->tyz; case 8: return &H->txz; case 9: return &H->txy;
    }
    return nullptr;
}
size_t dro_raw_size(dro_handle* H, int id) { std::vector<double>* a = H ? raw_array(H, id) : nullptr; return a ? a->size() : 0; }
int dro_get_raw(dro_handle* H, int id, double* dst, size_t n) {
    std::vector<double>* a = H ? raw_array(H, id) : nullptr;
    if (!a || !dst || n != a->size() || a->empty()) return DRO_ERR_ARG;
    std::memcpy(dst, a->data(), n * sizeof(double));
    return DRO_OK;
}
int dro_set_raw(dro_handle* H, int id, const double* src, size_t n) {
    std::vector<double>* a = H ? raw_array(H, id) : nullptr;
    if (!a || !src || n != a->size() || a->empty()) return DRO_ERR_ARG;
    std::memcpy(a->data(), src, n * sizeof(double));
    return DRO_OK;
}

const char* dro_last_error(dro_handle* H) { return H ? H->err.c_str() : "null handle"; }

void dro_destroy(dro_handle* H) { delete H; }

} /* extern "C" */
