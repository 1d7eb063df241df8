"""Pins of the nodal-projection oracle (oracle/nodal_oracle.c, readings N1..N10 in its header).

The paper prints nothing for this path (P:63 names the method only), so every pin is a closed form, an invariant,
brute force or an independent assembly:
  NP1 the V-cycle result at rel_tol = 1e-13 equals a dense direct solve (numpy) of the matrix assembled column by
      column, four boundary sets incl. spherical geometry;
  NP2 the operator equals an independent finite-element assembly (1-D element matrices, numpy kron, scipy sparse), is
      symmetric, has zero row sums away from OUTFLOW nodes, and is the textbook 27-point Q1 stencil for sigma = 1;
  NP3 manufactured solution: second-order convergence of phi (WALL and OUTFLOW);
  NP4 D = -G^T, and the correction equals numpy's cell-mean gradient;
  NP5 constant-coefficient periodic Fourier mode: eigenvalue in closed form, phi = rhs / lambda;
  NP6 restriction and prolongation equal (1/8) P^T and P built from 1-D interpolation matrices (scipy kron);
  NP7 convergence factors of the V(2,2) Jacobi cycle, h-independent;
  NP8 the approximate-projection identity D(beta0 U_new) - M beta0 S - m w = rhs - D(sigma G phi) and its O(h^2) size;
  NP9 scaling laws (rho -> c rho: phi -> c phi, U_new unchanged; beta0 -> c beta0: both unchanged).
"""
import numpy as np
import pytest
import scipy.sparse as sp

from paper_1910_12979_b200 import workloads as W

PER, WALL, OUT = W.PERIODIC, W.WALL, W.OUTFLOW


@pytest.fixture(scope="module")
def N(oracle):
    from oracle import nodal_oracle
    nodal_oracle.lib()
    return nodal_oracle


def structs(N, wl, **mg_kw):
    g = N.make_grid(wl.n, wl.dx, wl.bc_lo, wl.bc_hi)
    b = N.make_base(wl.geometry, wl.nr, wl.dr, wl.center)
    kw = dict(nu_pre=2, nu_post=2, max_cycles=100, rel_tol=wl.rel_tol)
    kw.update(mg_kw)
    return g, b, N.make_mg(**kw)


def project(N, wl, **mg_kw):
    g, b, mg = structs(N, wl, **mg_kw)
    u, v, w = W.cell_centred(wl)
    status, phi, st = N.project(g, b, mg, wl.beta0, wl.rho0, wl.rho, u, v, w, wl.S)
    return dict(status=status, phi=phi, u=u, v=v, w=w, stats=st, g=g, b=b)


def unknown_mask(N, g):
    return N.node_kind(g) == 0


BC_SETS = [
    ((PER, PER, PER), (PER, PER, PER)),
    ((PER, PER, WALL), (PER, PER, WALL)),
    ((OUT, OUT, OUT), (OUT, OUT, OUT)),
    ((OUT, WALL, PER), (WALL, OUT, PER)),
    ((WALL, WALL, WALL), (WALL, WALL, WALL)),
]


# ---- independent finite-element assembly ---------------------------------------------------------------------

def fe_matrix(sig, h, bc_lo, bc_hi):
    """-L V-scaled: A[a, b] = (1/V) sum_c sigma_c int_c grad psi_a . grad psi_b over ALL (nx+1)(ny+1)(nz+1) nodes,
    periodic duplicates folded onto their images.  1-D linear-element matrices combined by Kronecker products."""
    nz, ny, nx = sig.shape
    nn = (nx + 1, ny + 1, nz + 1)
    K1 = [np.array([[1.0, -1.0], [-1.0, 1.0]]) / hd for hd in h]
    M1 = [np.array([[2.0, 1.0], [1.0, 2.0]]) * hd / 6.0 for hd in h]
    Ke = (np.kron(M1[2], np.kron(M1[1], K1[0])) + np.kron(M1[2], np.kron(K1[1], M1[0])) +
          np.kron(K1[2], np.kron(M1[1], M1[0]))) / (h[0] * h[1] * h[2])
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")

    def nid(ii, jj, kk):
        if bc_lo[0] == PER: ii = ii % nx
        if bc_lo[1] == PER: jj = jj % ny
        if bc_lo[2] == PER: kk = kk % nz
        return (ii + nn[0] * (jj + nn[1] * kk)).ravel()
    rows, cols, vals = [], [], []
    for a in range(8):
        for b in range(8):
            rows.append(nid(i + (a & 1), j + ((a >> 1) & 1), k + (a >> 2)))
            cols.append(nid(i + (b & 1), j + ((b >> 1) & 1), k + (b >> 2)))
            vals.append((sig * Ke[a, b]).ravel())
    n_all = nn[0] * nn[1] * nn[2]
    return sp.csr_matrix((np.concatenate(vals), (np.concatenate(rows), np.concatenate(cols))), shape=(n_all, n_all))


def oracle_matrix(N, g, sig):
    """L restricted to the unknowns, column by column from the oracle's own operator."""
    mask = unknown_mask(N, g).ravel()
    idx = np.where(mask)[0]
    A = np.zeros((len(idx), len(idx)))
    e = np.zeros(N.node_shape(g))
    for q, a in enumerate(idx):
        e.flat[a] = 1.0
        A[:, q] = N.apply(g, sig, e).ravel()[idx]
        e.flat[a] = 0.0
    return A, idx


@pytest.mark.parametrize("bc", range(len(BC_SETS)))
def test_np2_operator_equals_independent_fe_assembly(N, bc):
    lo, hi = BC_SETS[bc]
    wl = W.mixed_bc_case(n=(6, 4, 8), bc_lo=lo, bc_hi=hi, seed=60 + bc)
    g, b, _ = structs(N, wl)
    rng = np.random.default_rng(bc)
    sig = np.exp(rng.uniform(-1, 1, size=wl.rho.shape))
    A, idx = oracle_matrix(N, g, sig)
    F = fe_matrix(sig, wl.dx, lo, hi).toarray()[np.ix_(idx, idx)]
    scale = np.abs(F).max()
    assert np.abs(A + F).max() <= 1e-13 * scale                      # L = -A_fe
    assert np.abs(A - A.T).max() <= 1e-13 * scale                    # symmetric
    if OUT not in lo + hi:
        assert np.abs(A.sum(axis=1)).max() <= 1e-12 * scale          # constants are in the null space
    # the diagonal the Jacobi sweep divides by
    d = N.diag(g, sig).ravel()[idx]
    assert np.allclose(d, np.diag(A), rtol=1e-13)
    # OUTFLOW nodes and periodic duplicates: the operator ignores what the array holds there
    phi = rng.standard_normal(N.node_shape(g))
    out1 = N.apply(g, sig, phi)
    junk = phi.copy()
    junk[N.node_kind(g) != 0] = 1e30
    assert np.array_equal(out1, N.apply(g, sig, junk))
    assert np.all(out1[N.node_kind(g) != 0] == 0.0)


def test_np2_textbook_q1_stencil(N):
    wl = W.config1(N=8)
    g = N.make_grid((8, 8, 8), (1.0, 1.0, 1.0), (WALL,) * 3, (WALL,) * 3)
    sig = np.ones((8, 8, 8))
    e = np.zeros(N.node_shape(g)); e[4, 4, 4] = 1.0
    col = N.apply(g, sig, e)[3:6, 3:6, 3:6]
    exp = np.empty((3, 3, 3))
    for dk in range(3):
        for dj in range(3):
            for di in range(3):
                nz_ = (dk != 1) + (dj != 1) + (di != 1)
                exp[dk, dj, di] = {0: -8.0 / 3.0, 1: 0.0, 2: 1.0 / 6.0, 3: 1.0 / 12.0}[nz_]
    assert np.allclose(col, exp, atol=1e-15)
    assert N.omega(g) == 1.0
    ga = N.make_grid((8, 8, 8), (1.0, 0.5, 0.25), (WALL,) * 3, (WALL,) * 3)     # stretched: omega lambda_max stays 3/2
    gd = np.array([1.0, 4.0, 16.0])
    assert N.omega(ga) == pytest.approx(gd.sum() / (3 * gd.max()), rel=1e-15)


@pytest.mark.parametrize("bc", range(len(BC_SETS)))
@pytest.mark.parametrize("geometry", [W.PLANAR, W.SPHERICAL])
def test_np1_vcycle_equals_dense_direct_solve(N, bc, geometry):
    lo, hi = BC_SETS[bc]
    wl = W.mixed_bc_case(n=(8, 8, 8), bc_lo=lo, bc_hi=hi, seed=70 + bc, geometry=geometry)
    wl.dx = (1.0 / 8, 1.0 / 8, 1.0 / 8)
    if geometry == W.PLANAR:
        wl.dr = wl.dx[2]
    wl.rel_tol = 1e-13
    r = project(N, wl)
    assert r["status"] == 0
    g, b = r["g"], r["b"]
    sig = N.sigma(g, b, wl.beta0, wl.rho)
    A, idx = oracle_matrix(N, g, sig)
    rhs = N.rhs(g, b, wl.beta0, *W.cell_centred(wl), wl.S)
    wgt = N.weights(g)
    singular = OUT not in lo + hi
    f = rhs.ravel()[idx].copy()
    if singular:
        m = f.sum() / wl.ncells
        assert r["stats"]["rhs_mean_removed"] == pytest.approx(m, rel=1e-10, abs=1e-14)
        f -= m * wgt.ravel()[idx]
        n = len(idx)
        B = np.zeros((n + 1, n + 1)); B[:n, :n] = A; B[:n, n] = 1.0; B[n, :n] = wgt.ravel()[idx]
        x = np.linalg.solve(B, np.concatenate([f, [0.0]]))[:n]           # zero w-weighted mean (N5)
    else:
        x = np.linalg.solve(A, f)
    got = r["phi"].ravel()[idx]
    assert np.linalg.norm(got - x) <= 1e-11 * np.linalg.norm(x)
    # periodic duplicates carry their image, OUTFLOW nodes 0
    kind = N.node_kind(g)
    assert np.all(r["phi"][kind == 1] == 0.0)
    if lo[0] == PER:
        assert np.array_equal(r["phi"][:, :, -1], r["phi"][:, :, 0])
    if lo[2] == PER:
        assert np.array_equal(r["phi"][-1], r["phi"][0])


def numpy_cell_gradient(phi, h):
    """cell-mean gradient of a nodal array: mean of the 4 edge differences per axis (independent of the oracle)."""
    dx = (phi[:, :, 1:] - phi[:, :, :-1]) / h[0]
    gx = 0.25 * (dx[:-1, :-1] + dx[1:, :-1] + dx[:-1, 1:] + dx[1:, 1:])
    dy = (phi[:, 1:, :] - phi[:, :-1, :]) / h[1]
    gy = 0.25 * (dy[:-1, :, :-1] + dy[1:, :, :-1] + dy[:-1, :, 1:] + dy[1:, :, 1:])
    dz = (phi[1:, :, :] - phi[:-1, :, :]) / h[2]
    gz = 0.25 * (dz[:, :-1, :-1] + dz[:, 1:, :-1] + dz[:, :-1, 1:] + dz[:, 1:, 1:])
    return gx, gy, gz


@pytest.mark.parametrize("bc", range(len(BC_SETS)))
def test_np4_divergence_is_minus_gradient_transposed(N, bc):
    lo, hi = BC_SETS[bc]
    wl = W.mixed_bc_case(n=(10, 6, 8), bc_lo=lo, bc_hi=hi, seed=80 + bc)
    g, b, _ = structs(N, wl)
    rng = np.random.default_rng(bc)
    kind = N.node_kind(g)
    phi = rng.standard_normal(N.node_shape(g))
    # a consistent nodal field: OUTFLOW nodes 0, periodic duplicates equal their image
    phi[kind == 1] = 0.0
    if lo[0] == PER: phi[:, :, -1] = phi[:, :, 0]
    if lo[1] == PER: phi[:, -1, :] = phi[:, 0, :]
    if lo[2] == PER: phi[-1, :, :] = phi[0, :, :]
    rho = np.exp(rng.uniform(-1, 1, size=wl.rho.shape))
    F = [rng.standard_normal(wl.rho.shape) for _ in range(3)]
    # G from the correction with U = 0: result = -(1/rho) G phi
    u, v, w = (np.zeros(wl.rho.shape) for _ in range(3))
    N.correct(g, rho, phi, u, v, w)
    gx, gy, gz = numpy_cell_gradient(phi, wl.dx)
    for got, ref in ((u, gx), (v, gy), (w, gz)):
        assert np.abs(got + ref / rho).max() <= 1e-13 * np.abs(ref / rho).max()
    # D from the rhs with beta0 = 1, S = 0:  <phi, D F>_unknowns = -<G phi, F>_cells
    ones = np.ones(wl.nr)
    DF = N.rhs(g, b, ones, *F, None)
    lhs = (phi * DF)[kind == 0].sum()
    rhs_ = -(gx * F[0] + gy * F[1] + gz * F[2]).sum()
    assert lhs == pytest.approx(rhs_, rel=1e-12)
    # M: the source term is the mean of beta0 S over the cells around a node (interior nodes: all 8)
    S = rng.standard_normal(wl.rho.shape)
    zero = np.zeros(wl.rho.shape)
    MS = -N.rhs(g, b, ones, zero, zero, zero, S)
    box = sum(S[dk:S.shape[0] - 1 + dk, dj:S.shape[1] - 1 + dj, di:S.shape[2] - 1 + di]
              for dk in (0, 1) for dj in (0, 1) for di in (0, 1)) / 8.0
    assert np.allclose(MS[1:-1, 1:-1, 1:-1], box, rtol=1e-13, atol=1e-15)
    # weights: (cells around the node) / 8; their sum over the unknowns is the cell count unless OUTFLOW nodes drop out
    wgt = N.weights(g)
    if OUT not in lo + hi:
        assert wgt.sum() == pytest.approx(wl.ncells, rel=1e-14)


def test_np5_fourier_mode(N):
    n = 16
    h = 1.0 / n
    g = N.make_grid((n, n, n), (h, h, h), (PER,) * 3, (PER,) * 3)
    sig = np.ones((n, n, n))
    x = np.arange(n + 1) * h
    kx, ky, kz = 3, 1, 2
    mode = (np.cos(2 * np.pi * kz * x)[:, None, None] * np.cos(2 * np.pi * ky * x)[None, :, None] *
            np.cos(2 * np.pi * kx * x)[None, None, :])
    th = 2 * np.pi * np.array([kx, ky, kz]) / n
    s2, mm = np.sin(th / 2) ** 2, (2 + np.cos(th)) / 3
    lam = -(4 / h ** 2) * (s2[0] * mm[1] * mm[2] + mm[0] * s2[1] * mm[2] + mm[0] * mm[1] * s2[2])
    out = N.apply(g, sig, mode)
    m = unknown_mask(N, g)
    assert np.abs(out[m] - lam * mode[m]).max() <= 1e-11 * abs(lam)
    # V-cycles: phi = rhs / lambda
    mg = N.make_mg(rel_tol=1e-13)
    phi = np.zeros(N.node_shape(g))
    rhs = mode.copy(); rhs[~m] = 0.0
    for _ in range(30):
        N.vcycle(g, sig, rhs, phi, mg)
    assert np.abs(phi[m] - mode[m] / lam).max() <= 1e-10 * abs(1 / lam)


def prolong_1d(nc, bc_lo, bc_hi):
    """fine nodes (2 nc + 1) x coarse nodes (nc + 1), node rules of N4 folded in."""
    nf = 2 * nc
    P = np.zeros((nf + 1, nc + 1))
    for I in range(nc + 1):
        P[2 * I, I] = 1.0
    for I in range(nc):
        P[2 * I + 1, I] = 0.5; P[2 * I + 1, I + 1] = 0.5
    if bc_lo == PER:                       # node n is node 0
        P[:, 0] += P[:, nc]; P[:, nc] = 0.0
        P[nf, :] = 0.0
    else:
        if bc_lo == OUT: P[:, 0] = 0.0; P[0, :] = 0.0
        if bc_hi == OUT: P[:, nc] = 0.0; P[nf, :] = 0.0
    return sp.csr_matrix(P)


@pytest.mark.parametrize("bc", range(len(BC_SETS)))
def test_np6_transfer_operators(N, bc):
    lo, hi = BC_SETS[bc]
    wl = W.mixed_bc_case(n=(12, 8, 16), bc_lo=lo, bc_hi=hi, seed=90 + bc)
    g, _, _ = structs(N, wl)
    P = sp.kron(prolong_1d(8, lo[2], hi[2]), sp.kron(prolong_1d(4, lo[1], hi[1]), prolong_1d(6, lo[0], hi[0]))).tocsr()
    rng = np.random.default_rng(bc)
    gc = N.M.coarsen_grid(g)
    ec = rng.standard_normal(N.node_shape(gc))
    fine = rng.standard_normal(N.node_shape(g))
    ref = fine.copy().ravel() + P @ ec.ravel()
    got = fine.copy()
    N.prolong_add(g, ec, got)
    m = unknown_mask(N, g).ravel()
    assert np.abs(got.ravel()[m] - ref[m]).max() <= 1e-14 * np.abs(ref).max()
    assert np.array_equal(got.ravel()[~m], fine.ravel()[~m])          # only unknowns are touched
    r = rng.standard_normal(N.node_shape(g))
    r[N.node_kind(g) != 0] = 0.0
    rc = N.restrict(g, r)
    refc = (P.T @ r.ravel()) / 8.0
    mc = unknown_mask(N, gc).ravel()
    assert np.abs(rc.ravel()[mc] - refc[mc]).max() <= 1e-14 * np.abs(refc).max()
    assert np.all(rc.ravel()[~mc] == 0.0)
    # coarse sigma: mean of the 8 children
    sig = np.exp(rng.uniform(-1, 1, size=wl.rho.shape))
    _, sc = N.coarsen_sigma(g, sig)
    assert np.allclose(sc, sig.reshape(8, 2, 4, 2, 6, 2).mean(axis=(1, 3, 5)), rtol=1e-15)


@pytest.mark.parametrize("kind", ["wall", "outflow"])
def test_np3_manufactured_solution_second_order(N, kind):
    errs = []
    for n in (8, 16, 32):
        h = 1.0 / n
        bcv = WALL if kind == "wall" else OUT
        g = N.make_grid((n, n, n), (h, h, h), (bcv,) * 3, (bcv,) * 3)
        b = N.make_base(W.PLANAR, n, h)
        xc = (np.arange(n) + 0.5) * h
        xn = np.arange(n + 1) * h
        Z, Y, X = np.meshgrid(xc, xc, xc, indexing="ij")
        Zn, Yn, Xn = np.meshgrid(xn, xn, xn, indexing="ij")
        beta0 = np.exp(-xc)                                     # beta0(z) sampled at the profile points = cell centres
        f = np.cos if kind == "wall" else np.sin
        df = (lambda t: -np.sin(t)) if kind == "wall" else np.cos
        pe = lambda x, y, z: f(np.pi * x) * f(2 * np.pi * y) * f(np.pi * z)
        rho = 1.0 + 0.3 * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y) * np.cos(np.pi * Z)
        sig = np.exp(-Z) / rho
        # -div(sigma grad phi_e) = beta0 S at cell centres (sigma = beta0/rho, analytic derivatives)
        fx, fy, fz = f(np.pi * X), f(2 * np.pi * Y), f(np.pi * Z)
        px, py, pz = np.pi * df(np.pi * X) * fy * fz, 2 * np.pi * fx * df(2 * np.pi * Y) * fz, np.pi * fx * fy * df(np.pi * Z)
        lap = -(np.pi ** 2 + 4 * np.pi ** 2 + np.pi ** 2) * fx * fy * fz
        rx = 0.3 * 2 * np.pi * np.cos(2 * np.pi * X) * np.cos(2 * np.pi * Y) * np.cos(np.pi * Z)
        ry = -0.3 * 2 * np.pi * np.sin(2 * np.pi * X) * np.sin(2 * np.pi * Y) * np.cos(np.pi * Z)
        rz = -0.3 * np.pi * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y) * np.sin(np.pi * Z)
        sx, sy, sz = -sig * rx / rho, -sig * ry / rho, -sig - sig * rz / rho
        S = -(sig * lap + sx * px + sy * py + sz * pz) / np.exp(-Z)
        zero = np.zeros((n, n, n))
        mg = N.make_mg(rel_tol=1e-12)
        st, phi, stats = N.project(g, b, mg, beta0, beta0, rho, zero.copy(), zero.copy(), zero.copy(), S)
        assert st == 0
        ex = pe(Xn, Yn, Zn)
        if kind == "wall":
            ex = ex - N.weighted_mean(g, ex)
        errs.append(np.abs(phi - ex).max())
    assert errs[0] / errs[1] > 3.3 and errs[1] / errs[2] > 3.6, errs


@pytest.mark.parametrize("name,bound", [("1", 0.15), ("2", 0.15), ("3N", 0.27), ("3D", 0.22), ("4N", 0.42), ("4D", 0.36)])
def test_np7_convergence_factor(N, name, bound):
    fac = {}
    for n in (16, 32):
        wl = W.by_name(name, n)
        r = project(N, wl)
        assert r["status"] == 0
        h = r["stats"]["res_history"]
        fac[n] = (h[-1] / h[1]) ** (1.0 / (len(h) - 2))
        assert h[-1] <= 1e-10
    assert fac[32] <= bound, fac
    assert fac[32] <= 1.6 * fac[16] + 0.05, fac                      # h-independent


def test_np8_approximate_projection_identity(N):
    sizes = []
    for n in (16, 32):
        wl = W.config2(N=n)
        # smooth data so that the O(h^2) size of the defect is visible
        xc = (np.arange(n) + 0.5) / n
        Z, Y, X = np.meshgrid(xc, xc, xc, indexing="ij")
        wl.rho = wl.rho0[:, None, None] * (1.0 + 0.1 * np.sin(2 * np.pi * X) * np.sin(2 * np.pi * Y) * np.cos(np.pi * Z))
        uc = np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y) * np.sin(np.pi * Z)
        vc = np.cos(2 * np.pi * X) * np.sin(2 * np.pi * Y) * np.sin(np.pi * Z)
        wc = np.sin(2 * np.pi * X + 1.0) * np.sin(2 * np.pi * Y) * np.sin(np.pi * Z)
        g, b, mg = structs(N, wl, rel_tol=1e-12)
        un, vn, wn = uc.copy(), vc.copy(), wc.copy()
        st, phi, stats = N.project(g, b, mg, wl.beta0, wl.rho0, wl.rho, un, vn, wn, wl.S)
        assert st == 0
        rhs = N.rhs(g, b, wl.beta0, uc, vc, wc, wl.S)
        wgt = N.weights(g)
        m = stats["rhs_mean_removed"]
        c = N.constraint(g, b, wl.beta0, un, vn, wn, wl.S) - m * wgt
        # D(sigma G phi) with the numpy gradient and the oracle's D (beta0 = 1)
        sig = N.sigma(g, b, wl.beta0, wl.rho)
        gx, gy, gz = numpy_cell_gradient(phi, wl.dx)
        DsG = N.rhs(g, b, np.ones(wl.nr), sig * gx, sig * gy, sig * gz, None)
        ref = (rhs - m * wgt) - DsG
        mask = unknown_mask(N, g)
        assert np.abs(c - ref)[mask].max() <= 1e-12 * np.abs(rhs).max()
        sizes.append(np.abs(c)[mask].max() / np.abs(rhs - m * wgt)[mask].max())
    assert sizes[1] < 0.4 * sizes[0], sizes                          # the projection is approximate to O(h^2)


def test_np9_scaling_laws(N):
    wl = W.config3(N=16, variant="D")
    a = project(N, wl, rel_tol=1e-12)
    wl2 = W.config3(N=16, variant="D"); wl2.rho = wl2.rho * 7.0
    b = project(N, wl2, rel_tol=1e-12)
    assert np.linalg.norm(b["phi"] - 7.0 * a["phi"]) <= 1e-10 * np.linalg.norm(7.0 * a["phi"])
    assert np.linalg.norm(b["u"] - a["u"]) <= 1e-10 * np.linalg.norm(a["u"])
    wl3 = W.config3(N=16, variant="D"); wl3.beta0 = wl3.beta0 * 3.0
    c = project(N, wl3, rel_tol=1e-12)
    assert np.linalg.norm(c["phi"] - a["phi"]) <= 1e-10 * np.linalg.norm(a["phi"])
    assert np.linalg.norm(c["w"] - a["w"]) <= 1e-10 * np.linalg.norm(a["w"])


def test_nodal_oracle_thread_count_independent(N):
    wl = W.config2(N=16)
    n0 = N.M.num_threads()
    N.M.set_num_threads(1)
    a = project(N, wl)
    N.M.set_num_threads(max(2, n0))
    b = project(N, wl)
    N.M.set_num_threads(n0)
    assert np.array_equal(a["phi"], b["phi"]) and np.array_equal(a["u"], b["u"])
    assert a["stats"]["res_history"] == b["stats"]["res_history"]
