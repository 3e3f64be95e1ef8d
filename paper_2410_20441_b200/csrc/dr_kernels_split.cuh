// dr_kernels_split.cuh -- the PT iteration as two plain kernels (stress update, then velocity update), one
// thread per node, in place.  This is the unfused BASELINE: 31 doubles of HBM traffic
// per voxel-iteration against 20 for the fused kernel; kept selectable (DR_KERNEL = 1) as the A/B reference
// for the ncu evidence and as a second implementation for the parity tests.
#pragma once
#include "dr_kernels_aux.cuh"

// d v_a / d x_b (times h) at an edge whose index along b is e in [0,n]: central inside, one-sided with the
// affine wall value on the boundary (ghost rule, SURVEY O6 T / Reading R5)
__device__ __forceinline__ double dr_dshear(double v_hi, double v_lo, int e, int n, double u0_wall) {
    if (e == 0) return 2.0 * (v_hi - u0_wall);
    if (e == n) return 2.0 * (u0_wall - v_lo);
    return v_hi - v_lo;
}

// Eq. 12-13 with the relaxation term implicit: s <- (s + theta * Hooke(grad v)) / (1 + theta)
// FORM 1 (displacement form): the stresses are Hooke's law of the displacement itself (no relaxation).
// V = buffer whose velocity/displacement fields are read, F = buffer whose stress fields are updated.
template <int GAVG, int FORM>
__global__ void __launch_bounds__(256)
k_stress_split(DrLayout L, DrPT P, DrConstFields V, DrFields F, const double* __restrict__ Kp, const double* __restrict__ Gp) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    int j = blockIdx.y * blockDim.y + threadIdx.y;
    int k = blockIdx.z;
    const int nx = L.nx, ny = L.ny, nz = L.nz;
    if (i > nx || j > ny) return;
    const long long sy = L.sy, sz = L.sz;
    const long long q = L.origin + i + sy * j + sz * k;
    const double* vx = V.f[F_VX];
    const double* vy = V.f[F_VY];
    const double* vz = V.f[F_VZ];
    const double h = P.h, ih = P.inv_h, th = P.theta, ri = P.rinv;
    const bool ci = i < nx, cj = j < ny, ck = k < nz;
    if (ci && cj && ck) {
        double dxx = (vx[q + 1] - vx[q]) * ih, dyy = (vy[q + sy] - vy[q]) * ih, dzz = (vz[q + sz] - vz[q]) * ih;
        double div = dxx + dyy + dzz;
        double Kc = Kp[q], Gc = Gp[q];
        double lam_div = (Kc - 2.0 * Gc / 3.0) * div;
        if (FORM) {
            F.f[F_SXX][q] = lam_div + 2.0 * Gc * dxx;
            F.f[F_SYY][q] = lam_div + 2.0 * Gc * dyy;
            F.f[F_SZZ][q] = lam_div + 2.0 * Gc * dzz;
        } else {
            F.f[F_SXX][q] = (F.f[F_SXX][q] + th * (lam_div + 2.0 * Gc * dxx)) * ri;
            F.f[F_SYY][q] = (F.f[F_SYY][q] + th * (lam_div + 2.0 * Gc * dyy)) * ri;
            F.f[F_SZZ][q] = (F.f[F_SZZ][q] + th * (lam_div + 2.0 * Gc * dzz)) * ri;
        }
    }
    const bool bi = (i == 0 || i == nx), bj = (j == 0 || j == ny), bk = (k == 0 || k == nz);
    if (ck) {                                   // tau_xy at (i h, j h, (k+.5) h)
        double t = 0.0;
        if (!(bi || bj) || P.ghost_xy) {
            double z = (k + 0.5) * h;
            double a = dr_dshear(vx[q], vx[q - sy], j, ny, dr_u0(P, 0, i * h, j == 0 ? 0.0 : P.Ly, z));
            double b = dr_dshear(vy[q], vy[q - 1], i, nx, dr_u0(P, 1, i == 0 ? 0.0 : P.Lx, j * h, z));
            double Ge = dr_edge_mean<GAVG>(Gp[q - 1 - sy], Gp[q - sy], Gp[q - 1], Gp[q]);
            t = FORM ? Ge * ((a + b) * ih) : (F.f[F_TXY][q] + th * Ge * ((a + b) * ih)) * ri;
        }
        F.f[F_TXY][q] = t;
    }
    if (cj) {                                   // tau_xz at (i h, (j+.5) h, k h)
        double t = 0.0;
        if (!(bi || bk) || P.ghost_xz) {
            double y = (j + 0.5) * h;
            double a = dr_dshear(vx[q], vx[q - sz], k, nz, dr_u0(P, 0, i * h, y, k == 0 ? 0.0 : P.Lz));
            double b = dr_dshear(vz[q], vz[q - 1], i, nx, dr_u0(P, 2, i == 0 ? 0.0 : P.Lx, y, k * h));
            double Ge = dr_edge_mean<GAVG>(Gp[q - 1 - sz], Gp[q - sz], Gp[q - 1], Gp[q]);
            t = FORM ? Ge * ((a + b) * ih) : (F.f[F_TXZ][q] + th * Ge * ((a + b) * ih)) * ri;
        }
        F.f[F_TXZ][q] = t;
    }
    if (ci) {                                   // tau_yz at ((i+.5) h, j h, k h)
        double t = 0.0;
        if (!(bj || bk) || P.ghost_yz) {
            double x = (i + 0.5) * h;
            double a = dr_dshear(vy[q], vy[q - sz], k, nz, dr_u0(P, 1, x, j * h, k == 0 ? 0.0 : P.Lz));
            double b = dr_dshear(vz[q], vz[q - sy], j, ny, dr_u0(P, 2, x, j == 0 ? 0.0 : P.Ly, k * h));
            double Ge = dr_edge_mean<GAVG>(Gp[q - sy - sz], Gp[q - sz], Gp[q - sy], Gp[q]);
            t = FORM ? Ge * ((a + b) * ih) : (F.f[F_TYZ][q] + th * Ge * ((a + b) * ih)) * ri;
        }
        F.f[F_TYZ][q] = t;
    }
}

// Eq. 11 with Eq. 17: v <- v + (C~^2 h^2 / (theta H_node)) div(sigma) at interior face nodes;
// H_node = stiffest of the six springs in the node's stencil (Reading R3); nodes with H_node = 0 are skipped.
// RES: also the residual max-norm res = max |F| h / (H_node |eps0|), warp-shuffle + block
// reduction, one atomicMax per block on the bit pattern.
// FORM 1: w <- (1-theta) w + C~^2 h^2 F / H_node, u <- u + w; w lives in the sigma_aa slots of the state buffer U,
// the stresses are read from S.  FORM 0: U and S are the same buffer.
template <int GAVG, int RES, int FORM>
__global__ void __launch_bounds__(256)
k_velocity_split(DrLayout L, DrPT P, DrFields U, DrConstFields S, const double* __restrict__ Kp, const double* __restrict__ Gp,
                 unsigned long long* res_bits) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    int j = blockIdx.y * blockDim.y + threadIdx.y;
    int k = blockIdx.z;
    const int nx = L.nx, ny = L.ny, nz = L.nz;
    const long long sy = L.sy, sz = L.sz;
    const long long q = L.origin + i + sy * j + sz * k;
    const double ih = P.inv_h;
    double rmax = 0.0;
    bool rnan = false;
    if (i < nx && j < ny && k < nz) {
        const double* sxx = S.f[F_SXX];
        const double* syy = S.f[F_SYY];
        const double* szz = S.f[F_SZZ];
        const double* txy = S.f[F_TXY];
        const double* txz = S.f[F_TXZ];
        const double* tyz = S.f[F_TYZ];
        auto Hc = [&](long long s) { return Kp[s] + 4.0 * Gp[s] / 3.0; };
        auto Gxy = [&](long long s) { return dr_edge_mean<GAVG>(Gp[s - 1 - sy], Gp[s - sy], Gp[s - 1], Gp[s]); };
        auto Gxz = [&](long long s) { return dr_edge_mean<GAVG>(Gp[s - 1 - sz], Gp[s - sz], Gp[s - 1], Gp[s]); };
        auto Gyz = [&](long long s) { return dr_edge_mean<GAVG>(Gp[s - sy - sz], Gp[s - sz], Gp[s - sy], Gp[s]); };
        const double hq = Hc(q), gxy = Gxy(q), gxz = Gxz(q), gyz = Gyz(q);
        if (i >= 1) {
            double Fx = ((sxx[q] - sxx[q - 1]) + (txy[q + sy] - txy[q]) + (txz[q + sz] - txz[q])) * ih;
            double Hn = fmax(fmax(Hc(q - 1), hq), fmax(fmax(gxy, Gxy(q + sy)), fmax(gxz, Gxz(q + sz))));
            if (Hn > 0.0) {
                if (RES) { double r = fabs(Fx) / Hn; rnan |= !(r == r); rmax = fmax(rmax, r); }
                if (FORM) { double w = (1.0 - P.theta) * U.f[F_SXX][q] + P.c2t * P.theta / Hn * Fx; U.f[F_SXX][q] = w; U.f[F_VX][q] += w; }
                else U.f[F_VX][q] += P.c2t / Hn * Fx;
            }
        }
        if (j >= 1) {
            double Fy = ((txy[q + 1] - txy[q]) + (syy[q] - syy[q - sy]) + (tyz[q + sz] - tyz[q])) * ih;
            double Hn = fmax(fmax(Hc(q - sy), hq), fmax(fmax(gxy, Gxy(q + 1)), fmax(gyz, Gyz(q + sz))));
            if (Hn > 0.0) {
                if (RES) { double r = fabs(Fy) / Hn; rnan |= !(r == r); rmax = fmax(rmax, r); }
                if (FORM) { double w = (1.0 - P.theta) * U.f[F_SYY][q] + P.c2t * P.theta / Hn * Fy; U.f[F_SYY][q] = w; U.f[F_VY][q] += w; }
                else U.f[F_VY][q] += P.c2t / Hn * Fy;
            }
        }
        if (k >= 1) {
            double Fz = ((txz[q + 1] - txz[q]) + (tyz[q + sy] - tyz[q]) + (szz[q] - szz[q - sz])) * ih;
            double Hn = fmax(fmax(Hc(q - sz), hq), fmax(fmax(gxz, Gxz(q + 1)), fmax(gyz, Gyz(q + sy))));
            if (Hn > 0.0) {
                if (RES) { double r = fabs(Fz) / Hn; rnan |= !(r == r); rmax = fmax(rmax, r); }
                if (FORM) { double w = (1.0 - P.theta) * U.f[F_SZZ][q] + P.c2t * P.theta / Hn * Fz; U.f[F_SZZ][q] = w; U.f[F_VZ][q] += w; }
                else U.f[F_VZ][q] += P.c2t / Hn * Fz;
            }
        }
    }
    if (RES) {
        __shared__ unsigned long long sm[32];
        unsigned long long b = rnan ? 0x7ff8000000000000ull : (unsigned long long)__double_as_longlong(rmax * P.res_scale);
        b = dr_block_max_bits(b, sm);
        if (threadIdx.x == 0 && threadIdx.y == 0 && b != 0ull) atomicMax(res_bits, b);
    }
}
