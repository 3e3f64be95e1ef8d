"""Brute-force pin for the oracle: the *fixed point* of the PT iteration obtained without any iteration.

The converged state of O7 is the minimiser of the discrete elastic energy
    E(u) = h^3/2 * [ sum_cells  K tr(d)^2 + 2G |dev d|^2   +   sum_edges  w_e G_e gamma_e^2 ]
over the interior face nodes (wall-normal nodes held at the affine value), where w_e is the trapezoid weight of
the edge (1 interior, 1/2 on a face, 1/4 on a domain edge) for edges that carry stress and 0 for boundary edges
that are stress free, and gamma_e on boundary edges uses the one-sided ghost difference.  Here the energy
Hessian is assembled as a dense matrix with explicit loops and the linear system is solved with numpy.linalg --
no pseudo-time, no relaxation, no shared code with oracle/ (different formulation: energy / B^T D B).
Used only for tiny grids (n <= 6).
"""
import numpy as np


def _clamp(a, n):
    return min(max(a, 0), n - 1)


def _hmean(vals):
    if any(v == 0.0 for v in vals):
        return 0.0
    return len(vals) / sum(1.0 / v for v in vals)


def effective_column(K, G, lc, eps0=1e-4, h=1.0, bc_mode=0):
    """K,G: (nz,ny,nx).  Returns the 6 volume-averaged stresses / eps0 (Voigt xx,yy,zz,yz,xz,xy)."""
    nz, ny, nx = K.shape
    n = (nx, ny, nz)
    D = np.zeros((3, 3))
    D[{0: (0, 0), 1: (1, 1), 2: (2, 2), 3: (1, 2), 4: (0, 2), 5: (0, 1)}[lc]] = eps0

    def u0(a, pos):
        return float(D[a] @ np.asarray(pos, dtype=float))

    # --- dof numbering: component a lives on faces normal to a
    shapes = [(nx + 1, ny, nz), (nx, ny + 1, nz), (nx, ny, nz + 1)]
    offs = np.cumsum([0] + [s[0] * s[1] * s[2] for s in shapes])
    ndof = offs[-1]

    def dof(a, idx):
        s = shapes[a]
        return offs[a] + idx[0] + s[0] * (idx[1] + s[1] * idx[2])

    def node_pos(a, idx):
        pos = [(idx[b] + 0.5) * h for b in range(3)]
        pos[a] = idx[a] * h
        return pos

    fixed = np.zeros(ndof, dtype=bool)
    uval = np.zeros(ndof)
    for a in range(3):
        s = shapes[a]
        for k in range(s[2]):
            for j in range(s[1]):
                for i in range(s[0]):
                    idx = (i, j, k)
                    d = dof(a, idx)
                    uval[d] = u0(a, node_pos(a, idx))       # affine everywhere (initial guess, irrelevant for free)
                    if idx[a] == 0 or idx[a] == n[a]:
                        fixed[d] = True

    rows = []      # each: (dict dof->coef, const, weight_energy, kind, avg_weight)
    # cells: three normal strains, coupled through K and G
    A = np.zeros((ndof, ndof))
    rhs = np.zeros(ndof)       # gradient constant part: E = 1/2 u A u + rhs.u
    cell_rows = []
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                c = (i, j, k)
                Kc, Gc = K[k, j, i], G[k, j, i]
                lam = Kc - 2.0 * Gc / 3.0
                Cn = np.array([[lam + 2 * Gc, lam, lam], [lam, lam + 2 * Gc, lam], [lam, lam, lam + 2 * Gc]])
                pairs = []
                for a in range(3):
                    hi = list(c); hi[a] += 1
                    pairs.append((dof(a, tuple(hi)), dof(a, c)))
                cell_rows.append((pairs, Cn))
                for a in range(3):
                    for b in range(3):
                        for (da, sa) in ((pairs[a][0], 1.0 / h), (pairs[a][1], -1.0 / h)):
                            for (db, sb) in ((pairs[b][0], 1.0 / h), (pairs[b][1], -1.0 / h)):
                                A[da, db] += Cn[a, b] * sa * sb

    # edges: family (a,b) with c the edge direction; voigt index: (1,2)->3, (0,2)->4, (0,1)->5
    edge_rows = []
    for (a, b, voigt) in ((1, 2, 3), (0, 2, 4), (0, 1, 5)):
        cdir = 3 - a - b
        rng = [None, None, None]
        rng[a] = range(n[a] + 1); rng[b] = range(n[b] + 1); rng[cdir] = range(n[cdir])
        for k in rng[2]:
            for j in rng[1]:
                for i in rng[0]:
                    e = (i, j, k)
                    on_a = e[a] == 0 or e[a] == n[a]
                    on_b = e[b] == 0 or e[b] == n[b]
                    bnd = on_a or on_b
                    enabled = (not bnd) or bc_mode == 1 or voigt == lc
                    # modulus: harmonic mean of the 4 cells round the edge, replicate padded
                    cells = []
                    for sa in (-1, 0):
                        for sb in (-1, 0):
                            cc = list(e); cc[a] = _clamp(e[a] + sa, n[a]); cc[b] = _clamp(e[b] + sb, n[b])
                            cells.append(G[cc[2], cc[1], cc[0]])
                    Ge = _hmean(cells)
                    w = (0.5 if on_a else 1.0) * (0.5 if on_b else 1.0)
                    if not enabled:
                        edge_rows.append((voigt, {}, 0.0, 0.0, w))
                        continue
                    coef = {}
                    const = 0.0
                    # gamma = d v_a / d x_b + d v_b / d x_a
                    for (comp, dirn) in ((a, b), (b, a)):
                        # v_comp nodes neighbouring the edge in direction dirn: index e[dirn]-1 and e[dirn]
                        lo = list(e); lo[dirn] = e[dirn] - 1
                        hi = list(e)
                        wall = list(node_pos(comp, hi)); wall[dirn] = e[dirn] * h   # the wall point
                        # node_pos gives (idx+.5)h in non-normal directions: for direction dirn we overwrote it
                        if e[dirn] == 0:
                            d = dof(comp, tuple(hi))
                            coef[d] = coef.get(d, 0.0) + 2.0 / h
                            const += -2.0 / h * u0(comp, wall)
                        elif e[dirn] == n[dirn]:
                            d = dof(comp, tuple(lo))
                            coef[d] = coef.get(d, 0.0) - 2.0 / h
                            const += 2.0 / h * u0(comp, wall)
                        else:
                            d1 = dof(comp, tuple(hi)); d0 = dof(comp, tuple(lo))
                            coef[d1] = coef.get(d1, 0.0) + 1.0 / h
                            coef[d0] = coef.get(d0, 0.0) - 1.0 / h
                    edge_rows.append((voigt, coef, const, Ge, w))
                    for da, ca in coef.items():
                        rhs[da] += w * Ge * ca * const
                        for db, cb in coef.items():
                            A[da, db] += w * Ge * ca * cb

    free = ~fixed
    # drop free dofs that no spring touches (all-void neighbourhood)
    dead = free & (np.abs(A).sum(axis=1) == 0)
    free = free & ~dead
    u = uval.copy()
    b = -(A[np.ix_(free, fixed)] @ u[fixed]) - rhs[free]
    u[free] = np.linalg.solve(A[np.ix_(free, free)], b)

    N = nx * ny * nz
    avg = np.zeros(6)
    for pairs, Cn in cell_rows:
        d = np.array([(u[p[0]] - u[p[1]]) / h for p in pairs])
        avg[:3] += Cn @ d
    for voigt, coef, const, Ge, w in edge_rows:
        gam = const + sum(cf * u[d] for d, cf in coef.items())
        avg[voigt] += w * Ge * gam
    return avg / N / eps0


def effective_C(K, G, eps0=1e-4, h=1.0, bc_mode=0):
    C = np.zeros((6, 6))
    for lc in range(6):
        C[:, lc] = effective_column(K, G, lc, eps0, h, bc_mode)
    return C
