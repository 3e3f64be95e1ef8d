// dr_layout.cuh -- HBM data layout and per-launch parameter blocks shared by all kernels of libdr.
//
// Every one of the 9 state fields (x2 ping-pong buffers) and the 2 modulus fields lives on the SAME padded
// box of PX*PY*PZ doubles, so one linear offset q addresses the node (i,j,k) of every field:
//     q(i,j,k) = origin + i + PX*j + PX*PY*k,   origin = OX + PX*(1 + PY)
// Logical node ranges (staggered grid, sec. 3.3): cells [0,nx), faces/edges up to nx inclusive; the box
// additionally holds a halo: OX = 17 doubles to the left in x, one node below in y and z, and at least one
// node above in x, y, z.  OX is odd so that the TMA boxes of the fused kernel, which start one node left of
// an even tile origin (i0 - 1), begin at an even element = 16-byte aligned address (TMA faults otherwise);
// PX is a multiple of 16 so that every row starts on a 128-byte line.
// Halo content: state fields 0 (never written), moduli replicate-padded (mirror image of the nearest cell,
// Reading R4), so kernels need no index clamping.
#pragma once
#include <cstddef>
#include <cstdint>

#define DR_OX 17

struct DrLayout {
    int nx, ny, nz;
    int PX, PY, PZ;
    long long sy, sz;      // strides in doubles: PX, PX*PY
    long long origin;      // offset of logical node (0,0,0)
    long long count;       // PX*PY*PZ doubles per field
};

static inline int dr_round_up(int a, int m) { return (a + m - 1) / m * m; }

static inline DrLayout dr_make_layout(int nx, int ny, int nz) {
    DrLayout L;
    L.nx = nx; L.ny = ny; L.nz = nz;
    L.PX = dr_round_up(DR_OX + nx + 2, 16);     // i in [-17, nx+1]
    if (L.PX % 64 == 0) L.PX += 16;              // keep the row pitch off multiples of 512 B
    L.PY = ny + 3;                               // j in [-1, ny+1]
    L.PZ = nz + 3;                               // k in [-1, nz+1]
    L.sy = L.PX;
    L.sz = (long long)L.PX * L.PY;
    L.origin = DR_OX + L.sy + L.sz;
    L.count = L.sz * L.PZ;
    return L;
}

// field order of the public API (dr_get_field): vx vy vz sxx syy szz tyz txz txy
enum { F_VX = 0, F_VY, F_VZ, F_SXX, F_SYY, F_SZZ, F_TYZ, F_TXZ, F_TXY, F_COUNT };

struct DrFields { double* f[F_COUNT]; };
struct DrConstFields { const double* f[F_COUNT]; };

// Per-solve constants (Eq. 14-21):
//   theta = dt~/Dt = C~ St / n_max  (uniform because K~ = K(x), G~ = G(x), Reading R2)
//   rinv  = 1/(1+theta)             (implicit relaxation term of Eq. 12-13, Reading R14)
//   c2t   = C~^2 h^2 / theta        (Eq. 17: dt~/rho~ = c2t / H_node)
struct DrPT {
    double theta, rinv, c2t;
    double h, inv_h;
    double D[9];           // displacement gradient of the load case, row-major D[3*a+b]
    double Lx, Ly, Lz;
    double res_scale;      // h / |eps0|
    int ghost_yz, ghost_xz, ghost_xy;   // boundary edges of that shear component carry stress (ghost rule, O6 T)
};
