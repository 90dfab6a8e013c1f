"""Pins of the CPU oracle (oracle/tm_oracle.c) against what the paper's operator and the mathematics fix.

The paper prints no worked field values, so the oracle is pinned by properties P1-P12 of
DESIGN.md section 4: Clifford algebra of the declared basis, closed-form free-field plane-wave action
and eigenvalues (antiperiodic momenta), gauge covariance, gamma5-tau1 hermiticity, R R^{-1} = 1,
the dense 2^4 / 2^3x4 Schur-complement solve against the full operator (Eq. 2.2-2.4),
special cases (Wilson, decoupled flavors, kappa -> 0), parity structure, the location of the
antiperiodic sign, linearity and translation covariance.  Everything here runs on the CPU.
"""
import numpy as np
import pytest

import oracle
import synth_inputs as si

I = 1j
# The declared gamma_4-diagonal ("non-relativistic") representation, typed by hand.
G1 = np.array([[0, 0, 0, I], [0, 0, I, 0], [0, -I, 0, 0], [-I, 0, 0, 0]])
G2 = np.array([[0, 0, 0, 1], [0, 0, -1, 0], [0, -1, 0, 0], [1, 0, 0, 0]], dtype=complex)
G3 = np.array([[0, 0, I, 0], [0, 0, 0, -I], [-I, 0, 0, 0], [0, I, 0, 0]])
G4 = np.diag([1, 1, -1, -1]).astype(complex)
G5 = np.array([[0, 0, 1, 0], [0, 0, 0, 1], [1, 0, 0, 0], [0, 1, 0, 0]], dtype=complex)
GAM = [G1, G2, G3, G4]
TAU1 = np.array([[0, 1], [1, 0]], dtype=complex)
TAU3 = np.diag([1, -1]).astype(complex)

KAPPA = 0.1632


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def grid(a, dims):
    """[..., V, ...] with V on axis 1 -> [nf, T, Z, Y, X, ...]"""
    X, Y, Z, T = dims
    return a.reshape(a.shape[0], T, Z, Y, X, *a.shape[2:])


AXIS = {0: 4, 1: 3, 2: 2, 3: 1}     # mu -> axis of grid()


def apply_spin_flavor(m8, psi):
    """(spin (x) flavor) 8x8 matrix, index (f, s), on psi [2, V, 4, 3]."""
    m = m8.reshape(2, 4, 2, 4)
    return np.einsum("fsgr,gvrc->fvsc", m, psi)


def apply_spin(m4, psi):
    return np.einsum("sr,fvrc->fvsc", m4, psi)


def ip(a, b):
    return np.vdot(a, b)


PARAMS = [
    dict(mu=0.004, epsilon=0.0, twist_flavor=1),
    dict(mu=0.3, epsilon=0.0, twist_flavor=-1),
    dict(mu=0.15, epsilon=0.19, twist_flavor=0),
]


def nf_of(kw):
    return 2 if kw["twist_flavor"] == 0 else 1


# ---- P11: the basis -------------------------------------------------------------------------------

def test_p11_clifford_algebra_and_declared_basis():
    g = [oracle.gamma(i) for i in range(5)]
    for mu in range(4):
        assert np.allclose(g[mu], GAM[mu])
        assert np.allclose(g[mu], g[mu].conj().T)
        for nu in range(4):
            anti = g[mu] @ g[nu] + g[nu] @ g[mu]
            assert np.allclose(anti, 2 * np.eye(4) * (mu == nu))
        assert np.allclose(g[4] @ g[mu] + g[mu] @ g[4], 0)
    assert np.allclose(g[4], G1 @ G2 @ G3 @ G4)
    assert np.allclose(g[4], G5)
    assert np.allclose(g[3], np.diag(np.diag(g[3])))          # gamma_4 diagonal
    for mu in range(4):                                        # rank-2 projectors
        for s in (+1, -1):
            assert np.linalg.matrix_rank(np.eye(4) + s * g[mu]) == 2


# ---- P4: R R^{-1} = 1, R^dag = R(-a) --------------------------------------------------------------

@pytest.mark.parametrize("kw", PARAMS)
def test_p4_twist_inverse_and_dagger(kw):
    dims = (2, 2, 2, 4)
    p = oracle.params(dims, KAPPA, **kw)
    psi = si.spinor_field(dims, nf_of(kw), seed=11)
    for dag in (0, 1):
        r = oracle.twist(psi, p, inverse=0, dagger=dag)
        assert rel(oracle.twist(r, p, inverse=1, dagger=dag), psi) < 1e-14
        assert rel(oracle.twist(oracle.twist(psi, p, 1, dag), p, 0, dag), psi) < 1e-14
    phi = si.spinor_field(dims, nf_of(kw), seed=12)
    # <phi, R psi> = <R^dag phi, psi>
    assert abs(ip(phi, oracle.twist(psi, p, 0, 0)) - ip(oracle.twist(phi, p, 0, 1), psi)) < 1e-10
    # dagger is a -> -a
    kw2 = dict(kw, mu=-kw["mu"])
    p2 = oracle.params(dims, KAPPA, **kw2)
    assert rel(oracle.twist(psi, p, 0, 1), oracle.twist(psi, p2, 0, 0)) < 1e-15
    # closed-form action on a site: (1 + i a g5 tau3 + b tau1) with hand-typed g5, tau
    a, b = 2 * KAPPA * kw["mu"], 2 * KAPPA * kw["epsilon"]
    if nf_of(kw) == 2:
        m8 = np.eye(8) + I * a * np.kron(TAU3, G5) + b * np.kron(TAU1, np.eye(4))
        assert rel(oracle.twist(psi, p), apply_spin_flavor(m8, psi)) < 1e-14
    else:
        m4 = np.eye(4) + I * a * kw["twist_flavor"] * G5
        assert rel(oracle.twist(psi, p), apply_spin(m4, psi)) < 1e-14


def test_twist_inverse_singular_is_an_error():
    dims = (2, 2, 2, 2)
    # 1 + a^2 - b^2 = 0  with a = 0, b = 1  ->  eps = 1 / (2 kappa)
    p = oracle.params(dims, KAPPA, mu=0.0, epsilon=1.0 / (2 * KAPPA), twist_flavor=0)
    with pytest.raises(RuntimeError):
        oracle.twist(si.spinor_field(dims, 2, 1), p, inverse=1)


# ---- P2: free field, closed form ------------------------------------------------------------------

def momentum_matrix(pvec, kw):
    a, b = 2 * KAPPA * kw["mu"], 2 * KAPPA * kw["epsilon"]
    A = 1 - 2 * KAPPA * sum(np.cos(pvec))
    S = 2 * KAPPA * sum(np.sin(pvec[m]) * GAM[m] for m in range(4))
    if nf_of(kw) == 2:
        return (A * np.eye(8) + I * np.kron(np.eye(2), S) + I * a * np.kron(TAU3, G5)
                + b * np.kron(TAU1, np.eye(4)))
    return A * np.eye(4) + I * S + I * a * kw["twist_flavor"] * G5


@pytest.mark.parametrize("kw", PARAMS)
@pytest.mark.parametrize("tb", [-1, +1])
def test_p2_free_field_plane_waves(kw, tb):
    dims = (4, 6, 4, 8)
    X, Y, Z, T = dims
    nf = nf_of(kw)
    p = oracle.params(dims, KAPPA, t_boundary=tb, **kw)
    U = si.gauge_field(dims, 0, "unit")
    rng = np.random.default_rng(5)
    for n in [(1, 2, 3, 1), (0, 0, 0, 0), (3, 5, 1, 6)]:
        # antiperiodic time: p4 = (2 n4 + 1) pi / T  (periodic: 2 pi n4 / T)
        pvec = np.array([2 * np.pi * n[0] / X, 2 * np.pi * n[1] / Y, 2 * np.pi * n[2] / Z,
                         (2 * n[3] + 1) * np.pi / T if tb == -1 else 2 * np.pi * n[3] / T])
        xs = np.arange(X)[None, None, None, :]
        ys = np.arange(Y)[None, None, :, None]
        zs = np.arange(Z)[None, :, None, None]
        ts = np.arange(T)[:, None, None, None]
        phase = np.exp(I * (pvec[0] * xs + pvec[1] * ys + pvec[2] * zs + pvec[3] * ts)).reshape(-1)
        u = rng.standard_normal((nf, 4, 3)) + I * rng.standard_normal((nf, 4, 3))
        psi = phase[None, :, None, None] * u[:, None]
        mp = momentum_matrix(pvec, kw)
        if nf == 2:
            mu_ = np.einsum("fsgr,grc->fsc", mp.reshape(2, 4, 2, 4), u)
        else:
            mu_ = np.einsum("sr,frc->fsc", mp, u)
        expect = phase[None, :, None, None] * mu_[:, None]
        assert rel(oracle.mat(psi, U, p), expect) < 1e-13

        # eigenvalues in closed form
        a, b = 2 * KAPPA * kw["mu"], 2 * KAPPA * kw["epsilon"]
        A = 1 - 2 * KAPPA * sum(np.cos(pvec))
        s = 2 * KAPPA * np.sqrt(sum(np.sin(pvec) ** 2))
        ev = np.linalg.eigvals(mp)
        if nf == 2:
            closed = [A + sg * np.sqrt((b + sg2 * I * s) ** 2 - a * a + 0j)
                      for sg in (+1, -1) for sg2 in (+1, -1)]
        else:
            closed = [A + I * np.sqrt(s * s + a * a), A - I * np.sqrt(s * s + a * a)]
        for c in closed:
            assert np.min(np.abs(ev - c)) < 1e-12
        for e in ev:
            assert min(abs(e - c) for c in closed) < 1e-12
        # an eigenvector of M(p) times the plane wave is an eigenvector of the lattice operator
        w, v = np.linalg.eig(mp)
        uvec = v[:, 0].reshape(nf, 4)
        col = rng.standard_normal(3) + I * rng.standard_normal(3)
        psi = phase[None, :, None, None] * (uvec[:, None, :, None] * col[None, None, None, :])
        assert rel(oracle.mat(psi, U, p), w[0] * psi) < 1e-12


# ---- P3: gauge covariance -------------------------------------------------------------------------

@pytest.mark.parametrize("kw", PARAMS)
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 6, 8, 10)])
def test_p3_gauge_covariance(kw, dims):
    nf = nf_of(kw)
    V = si.volume(dims)
    p = oracle.params(dims, KAPPA, **kw)
    U = si.gauge_field(dims, 21, "haar")
    g = si.haar_su3(V, seed=22, stream=7)                      # [V, 3, 3]
    psi = si.spinor_field(dims, nf, 23)
    gg = grid(g[None], dims)[0]                                # [T, Z, Y, X, 3, 3]
    Ug = np.empty_like(U)
    for mu in range(4):
        gshift = np.roll(gg, -1, axis=AXIS[mu] - 1).reshape(V, 3, 3)   # g(x + mu)
        Ug[mu] = g @ U[mu] @ gshift.conj().transpose(0, 2, 1)
    gpsi = np.einsum("vcd,fvsd->fvsc", g, psi)
    for dag in (0, 1):
        lhs = oracle.mat(gpsi, Ug, p, dagger=dag)
        rhs = np.einsum("vcd,fvsd->fvsc", g, oracle.mat(psi, U, p, dagger=dag))
        assert rel(lhs, rhs) < 1e-13
    # a transposed or un-daggered link breaks it: sanity that the check has teeth
    bad = oracle.mat(gpsi, Ug.transpose(0, 1, 3, 2).copy(), p)
    assert rel(bad, np.einsum("vcd,fvsd->fvsc", g, oracle.mat(psi, U, p))) > 1e-2


# ---- P1: gamma5 (tau1) hermiticity, dagger definition ---------------------------------------------

@pytest.mark.parametrize("kw", PARAMS)
def test_p1_gamma5_tau1_hermiticity(kw):
    dims = (4, 4, 6, 4)
    nf = nf_of(kw)
    p = oracle.params(dims, KAPPA, **kw)
    U = si.gauge_field(dims, 31, "haar")
    psi, phi = si.spinor_field(dims, nf, 32), si.spinor_field(dims, nf, 33)
    # <phi, M psi> = <M^dag phi, psi>, M^dag = mat(dagger=1)
    assert abs(ip(phi, oracle.mat(psi, U, p)) - ip(oracle.mat(phi, U, p, dagger=1), psi)) < 1e-9
    assert abs(ip(phi, oracle.dhop(psi, U, p)) - ip(oracle.dhop(phi, U, p, dagger=1), psi)) < 1e-9
    # D_hop^dag = gamma5 D_hop gamma5
    assert rel(oracle.dhop(phi, U, p, dagger=1),
               apply_spin(G5, oracle.dhop(apply_spin(G5, phi), U, p))) < 1e-14
    if nf == 2:   # gamma5 tau1 M tau1 gamma5 = M^dag
        G = np.kron(TAU1, G5)
        lhs = apply_spin_flavor(G, oracle.mat(apply_spin_flavor(G, phi), U, p))
        assert rel(lhs, oracle.mat(phi, U, p, dagger=1)) < 1e-14
    else:         # gamma5 M(mu) gamma5 = M(-mu)^dag
        pm = oracle.params(dims, KAPPA, **dict(kw, mu=-kw["mu"]))
        lhs = apply_spin(G5, oracle.mat(apply_spin(G5, phi), U, p))
        assert rel(lhs, oracle.mat(phi, U, pm, dagger=1)) < 1e-14


# ---- P5: dense Schur complement on tiny lattices (Eq. 2.2-2.4) ------------------------------------

def dense(op, nf, V):
    n = nf * V * 12
    m = np.empty((n, n), dtype=complex)
    e = np.zeros(n, dtype=complex)
    for j in range(n):
        e[j] = 1
        m[:, j] = op(e.reshape(nf, V, 4, 3)).reshape(-1)
        e[j] = 0
    return m


@pytest.mark.parametrize("kw", PARAMS)
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (2, 2, 2, 4)])
def test_p5_dense_schur_solve_matches_full_operator(kw, dims):
    nf = nf_of(kw)
    V = si.volume(dims)
    p = oracle.params(dims, KAPPA, **kw)
    U = si.gauge_field(dims, 41, "haar")
    M = dense(lambda v: oracle.mat(v, U, p), nf, V)
    par = np.broadcast_to(oracle.site_parity(dims)[None, :, None, None], (nf, V, 4, 3)).reshape(-1)
    ev, od = np.nonzero(par == 0)[0], np.nonzero(par == 1)[0]

    psi = si.spinor_field(dims, nf, 42)
    b = (M @ psi.reshape(-1)).reshape(nf, V, 4, 3)
    assert rel(np.linalg.solve(M, b.reshape(-1)), psi.reshape(-1)) < 1e-11

    b_e, b_o = si.mask_parity(b, dims, 0), si.mask_parity(b, dims, 1)
    psi_e, psi_o = si.mask_parity(psi, dims, 0), si.mask_parity(psi, dims, 1)
    # RHS of (2.2): b_e + kappa D_eo R_oo^{-1} b_o
    rhs = b_e + KAPPA * si.mask_parity(oracle.dhop(oracle.twist(b_o, p, inverse=1), U, p), dims, 0)
    for typ in (oracle.ASYM, oracle.SYM):
        Mhat = dense(lambda v: oracle.matpc(v, U, p, typ), nf, V)
        assert np.abs(Mhat[np.ix_(od, ev)]).max() == 0        # writes even sites only
        assert np.abs(Mhat[:, od]).max() == 0                 # reads even sites only
        r = rhs if typ == oracle.ASYM else oracle.twist(rhs, p, inverse=1)
        # the paper's LHS applied to the true psi_e reproduces the derived RHS ...
        assert rel(oracle.matpc(psi_e, U, p, typ), r) < 1e-12
        # ... and solving the even-even system returns psi_e
        sol = np.linalg.solve(Mhat[np.ix_(ev, ev)], r.reshape(-1)[ev])
        assert rel(sol, psi.reshape(-1)[ev]) < 1e-10
    # (2.4): psi_o = R_oo^{-1} (b_o + kappa D_oe psi_e)
    assert rel(oracle.reconstruct_odd(psi_e, b_o, U, p), psi_o) < 1e-12
    # the RHS as literally printed (no kappa, minus sign) is NOT consistent with the kappa^2 LHS
    lit = b_e - si.mask_parity(oracle.dhop(oracle.twist(b_o, p, inverse=1), U, p), dims, 0)
    assert rel(oracle.matpc(psi_e, U, p, oracle.ASYM), lit) > 1e-2


# ---- P6: composite adjointness, C7 identities -----------------------------------------------------

@pytest.mark.parametrize("kw", PARAMS)
def test_p6_composite_adjoint_and_dagger_identities(kw):
    dims = (4, 4, 4, 6)
    nf = nf_of(kw)
    p = oracle.params(dims, KAPPA, **kw)
    U = si.gauge_field(dims, 51, "haar")
    psi = si.mask_parity(si.spinor_field(dims, nf, 52), dims, 0)
    phi = si.mask_parity(si.spinor_field(dims, nf, 53), dims, 0)
    # ASYM: the daggered composite IS the adjoint
    lhs = ip(phi, oracle.matpc(psi, U, p, oracle.ASYM))
    assert abs(lhs - ip(oracle.matpc(phi, U, p, oracle.ASYM, dagger=1), psi)) < 1e-9
    # SYM: adjoint = R^dag [daggered composite] R^dag^{-1}
    adj = oracle.twist(oracle.matpc(oracle.twist(phi, p, 1, 1), U, p, oracle.SYM, dagger=1), p, 0, 1)
    assert abs(ip(phi, oracle.matpc(psi, U, p, oracle.SYM)) - ip(adj, psi)) < 1e-9
    # kernel-level: dagger kernel = (gamma5 tau1) plain kernel (gamma5 tau1)  [nd];
    #               dagger kernel(mu) = gamma5 plain kernel(-mu) gamma5        [deg]
    x = si.mask_parity(si.spinor_field(dims, nf, 54), dims, 1)
    for kt in (oracle.A, oracle.A_XPAY, oracle.B, oracle.REC):
        d = oracle.kernel(psi, x, U, p, 1, 1, kt)
        if nf == 2:
            G = np.kron(TAU1, G5)
            e = apply_spin_flavor(G, oracle.kernel(apply_spin_flavor(G, psi), apply_spin_flavor(G, x),
                                                   U, p, 1, 0, kt))
        else:
            pm = oracle.params(dims, KAPPA, **dict(kw, mu=-kw["mu"]))
            e = apply_spin(G5, oracle.kernel(apply_spin(G5, psi), apply_spin(G5, x), U, pm, 1, 0, kt))
        assert rel(d, e) < 1e-13


# ---- P13 / P14: the adjoint and right-hand-side compositions (NEXT-1 rows) -------------------------------

@pytest.mark.parametrize("kw", PARAMS)
@pytest.mark.parametrize("typ", [0, 1])
def test_p13_matpc_adjoint_is_the_adjoint(kw, typ):
    dims = (4, 4, 4, 6)
    nf = nf_of(kw)
    p = oracle.params(dims, KAPPA, **kw)
    U = si.gauge_field(dims, 61, "haar")
    psi = si.mask_parity(si.spinor_field(dims, nf, 62), dims, 0)
    phi = si.mask_parity(si.spinor_field(dims, nf, 63), dims, 0)
    adj = oracle.matpc_adjoint(phi, U, p, typ)
    assert np.abs(si.mask_parity(adj, dims, 1)).max() == 0
    assert abs(ip(phi, oracle.matpc(psi, U, p, typ)) - ip(adj, psi)) < 1e-9 * abs(ip(phi, phi))
    if typ == oracle.ASYM:      # C7: the daggered two-launch composite is this adjoint
        assert rel(oracle.matpc(phi, U, p, oracle.ASYM, dagger=1), adj) < 1e-13
    else:                       # C7: it is NOT for SYM (the twist changes sides) ...
        assert rel(oracle.matpc(phi, U, p, oracle.SYM, dagger=1), adj) > 1e-4      # 7e-4 already at mu = 0.004
        # ... but conjugating with R^dag relates the two
        conj = oracle.twist(oracle.matpc(oracle.twist(phi, p, 1, 1), U, p, oracle.SYM, dagger=1), p, 0, 1)
        assert rel(conj, adj) < 1e-12


@pytest.mark.parametrize("kw", PARAMS)
def test_p14_rhs_preparation_against_the_full_operator(kw):
    """b = M psi with the FULL operator (pinned by P1-P3); then M^ psi_e must equal the prepared right-hand side and
    Eq. (2.4) must give back psi_o: ties prepare_rhs, matpc and reconstruct_odd to oracle.mat on a lattice with
    every extent different."""
    dims = (4, 6, 8, 10)
    nf = nf_of(kw)
    p = oracle.params(dims, KAPPA, **kw)
    U = si.gauge_field(dims, 71, "near_identity")
    psi = si.spinor_field(dims, nf, 72)
    b = oracle.mat(psi, U, p)
    psi_e, psi_o = si.mask_parity(psi, dims, 0), si.mask_parity(psi, dims, 1)
    for typ in (oracle.ASYM, oracle.SYM):
        rhs = oracle.prepare_rhs(b, U, p, typ)
        assert np.abs(si.mask_parity(rhs, dims, 1)).max() == 0
        assert rel(oracle.matpc(psi_e, U, p, typ), rhs) < 1e-12
    assert rel(oracle.reconstruct_odd(psi_e, si.mask_parity(b, dims, 1), U, p), psi_o) < 1e-12
    # the plain xpay / axpy forms are what their names say
    x = si.mask_parity(si.spinor_field(dims, nf, 73), dims, 0)
    got = oracle.hop_xpay(psi_o, x, U, p, 0, 0, -KAPPA * KAPPA)
    assert rel(got, x - KAPPA * KAPPA * si.mask_parity(oracle.dhop(psi_o, U, p), dims, 0)) < 1e-14
    # ... and pinned through the full operator (P2, P5 pin `mat`), not through their own formula:  M = R - kappa D_hop, so
    #   (M psi)_e = hop_xpay(psi_o, R psi_e; even, -kappa)   and, with b = M psi,   R psi_o = hop_xpay(psi_e, b_o; odd, +kappa)
    r_e = oracle.twist(psi_e, p, 0, 0)
    assert rel(oracle.hop_xpay(psi_o, r_e, U, p, 0, 0, -KAPPA), si.mask_parity(b, dims, 0)) < 1e-13
    r_o = oracle.twist(psi_o, p, 0, 0)
    assert rel(oracle.hop_xpay(psi_e, si.mask_parity(b, dims, 1), U, p, 1, 0, +KAPPA), r_o) < 1e-13
    # the fused D R^-1 forms are pinned the same way: Eq. 2.2 / 2.3 right-hand sides (P14's prepare_rhs, tied to b = M psi above)
    # and the first stage of the exact SYM adjoint (P13's matpc_adjoint)
    be, bo = si.mask_parity(b, dims, 0), si.mask_parity(b, dims, 1)
    assert rel(oracle.kernel_twist_in(bo, be, U, p, 0, 0, "AXPY"), oracle.prepare_rhs(b, U, p, oracle.ASYM)) < 1e-13
    assert rel(oracle.kernel_twist_in(bo, be, U, p, 0, 0, "REC"), oracle.prepare_rhs(b, U, p, oracle.SYM)) < 1e-13
    assert rel(oracle.kernel_twist_in(bo, be, U, p, 0, 0, "AXPY"), oracle.matpc(psi_e, U, p, oracle.ASYM)) < 1e-12
    t_o = oracle.kernel_twist_in(psi_e, None, U, p, 1, 1, "A")
    assert rel(oracle.hop_xpay(t_o, psi_e, U, p, 0, 1, -KAPPA * KAPPA), oracle.matpc_adjoint(psi_e, U, p, oracle.SYM)) < 1e-13
    # the daggered form is the adjoint of the plain one between the two parities: <phi_e, D_eo psi_o> = <D^dag_oe phi_e, psi_o>
    phi_e = si.mask_parity(si.spinor_field(dims, nf, 74), dims, 0)
    zero = np.zeros_like(psi)
    lhs = np.vdot(phi_e, oracle.hop_xpay(psi_o, zero, U, p, 0, 0, 1.0))
    rhs_ = np.vdot(oracle.hop_xpay(phi_e, zero, U, p, 1, 1, 1.0), psi_o)
    assert abs(lhs - rhs_) <= 1e-12 * abs(lhs)


# ---- P7 / P8: special cases -----------------------------------------------------------------------

def test_p7_wilson_and_decoupled_flavors():
    dims = (4, 4, 4, 6)
    U = si.gauge_field(dims, 61, "near_identity")
    psi2 = si.spinor_field(dims, 2, 62)
    # mu = eps = 0: M = 1 - kappa D_hop, same for both flavors
    p0 = oracle.params(dims, KAPPA, mu=0.0, epsilon=0.0, twist_flavor=0)
    p0d = oracle.params(dims, KAPPA, mu=0.0, epsilon=0.0, twist_flavor=1)
    out = oracle.mat(psi2, U, p0)
    for f in range(2):
        one = psi2[f:f + 1]
        assert rel(out[f:f + 1], one - KAPPA * oracle.dhop(one, U, p0d)) < 1e-14
        assert rel(out[f:f + 1], oracle.mat(one, U, p0d)) < 1e-15
    # eps = 0: the doublet is two independent degenerate operators with tau3 = +1 / -1
    pn = oracle.params(dims, KAPPA, mu=0.25, epsilon=0.0, twist_flavor=0)
    out = oracle.mat(psi2, U, pn)
    for f, tw in ((0, +1), (1, -1)):
        pd = oracle.params(dims, KAPPA, mu=0.25, epsilon=0.0, twist_flavor=tw)
        assert rel(out[f:f + 1], oracle.mat(psi2[f:f + 1], U, pd)) < 1e-15
        for kt in (oracle.A, oracle.A_XPAY, oracle.B, oracle.REC):
            kn = oracle.kernel(psi2, psi2, U, pn, 0, 0, kt)
            kd = oracle.kernel(psi2[f:f + 1], psi2[f:f + 1], U, pd, 0, 0, kt)
            assert rel(kn[f:f + 1], kd) < 1e-15


def test_p8_kappa_to_zero_is_local():
    dims = (4, 4, 4, 4)
    U = si.gauge_field(dims, 63, "haar")
    psi = si.spinor_field(dims, 2, 64)
    p = oracle.params(dims, 0.0, mu=0.15, epsilon=0.19, twist_flavor=0)
    assert rel(oracle.mat(psi, U, p), psi) < 1e-15            # a = b = 0 at kappa = 0
    # M = R - kappa D_hop for any kappa
    p = oracle.params(dims, KAPPA, mu=0.15, epsilon=0.19, twist_flavor=0)
    assert rel(oracle.mat(psi, U, p), oracle.twist(psi, p) - KAPPA * oracle.dhop(psi, U, p)) < 1e-14


# ---- P9: parity structure -------------------------------------------------------------------------

def test_p9_hop_connects_opposite_parities_only():
    dims = (4, 6, 4, 8)
    U = si.gauge_field(dims, 71, "haar")
    p = oracle.params(dims, KAPPA, mu=0.15, epsilon=0.19, twist_flavor=0)
    psi = si.spinor_field(dims, 2, 72)
    par = oracle.site_parity(dims)
    assert np.array_equal(par[si.parity_sites(dims, 0)], np.zeros(si.volume(dims) // 2, dtype=par.dtype))
    for q in (0, 1):
        out = oracle.dhop(si.mask_parity(psi, dims, q), U, p)
        assert np.abs(out[:, par == q]).max() == 0
        assert np.abs(out[:, par == 1 - q]).min() > 0
        tw = oracle.twist(si.mask_parity(psi, dims, q), p)
        assert np.abs(tw[:, par == 1 - q]).max() == 0


# ---- P10: unit links, constant spinor; where the antiperiodic sign sits ---------------------------

def test_p10_constant_field_and_time_boundary_sign():
    dims = (4, 4, 4, 6)
    X, Y, Z, T = dims
    U = si.gauge_field(dims, 0, "unit")
    rng = np.random.default_rng(3)
    u = rng.standard_normal((1, 4, 3)) + I * rng.standard_normal((1, 4, 3))
    psi = np.broadcast_to(u[:, None], (1, si.volume(dims), 4, 3)).copy()
    pp = oracle.params(dims, KAPPA, mu=0.0, t_boundary=+1)
    assert rel(oracle.dhop(psi, U, pp), 8 * psi) < 1e-15
    pa = oracle.params(dims, KAPPA, mu=0.0, t_boundary=-1)
    out = grid(oracle.dhop(psi, U, pa), dims)[0]              # [T, Z, Y, X, 4, 3]
    ref = grid(8 * psi, dims)[0]
    assert np.abs(out[1:T - 1] - ref[1:T - 1]).max() < 1e-14
    # t = T-1: the forward hop (1 - gamma_4) flips sign; t = 0: the backward hop (1 + gamma_4)
    fwd = np.einsum("sr,rc->sc", np.eye(4) - G4, u[0])
    bwd = np.einsum("sr,rc->sc", np.eye(4) + G4, u[0])
    assert np.abs(out[T - 1] - (8 * u[0] - 2 * fwd)).max() < 1e-14
    assert np.abs(out[0] - (8 * u[0] - 2 * bwd)).max() < 1e-14
    # daggered hop: projectors swap
    outd = grid(oracle.dhop(psi, U, pa, dagger=1), dims)[0]
    assert np.abs(outd[T - 1] - (8 * u[0] - 2 * bwd)).max() < 1e-14
    assert np.abs(outd[0] - (8 * u[0] - 2 * fwd)).max() < 1e-14


def test_p10b_single_hop_direction_and_link_orientation():
    """A delta source at y with only U_mu(y) non-trivial: (D_hop delta_y)(y - mu) = (1 - g_mu) U_mu(y - mu)...
    pins which link and which projector each of the two hops uses."""
    dims = (4, 4, 4, 4)
    X, Y, Z, T = dims
    V = si.volume(dims)
    U = si.gauge_field(dims, 81, "haar")
    p = oracle.params(dims, KAPPA, mu=0.0, t_boundary=+1)
    rng = np.random.default_rng(8)
    u = rng.standard_normal((4, 3)) + I * rng.standard_normal((4, 3))
    y = (1, 2, 3, 1)
    lex = lambda c: c[0] + X * (c[1] + Y * (c[2] + Z * c[3]))
    src = np.zeros((1, V, 4, 3), dtype=complex)
    src[0, lex(y)] = u
    out = oracle.dhop(src, U, p)[0]
    nz = 0
    for mu in range(4):
        ym = list(y); ym[mu] = (y[mu] - 1) % dims[mu]
        yp = list(y); yp[mu] = (y[mu] + 1) % dims[mu]
        # site x = y - mu sees psi(x + mu) = u through the forward hop: (1 - g_mu) U_mu(x) u
        e = np.einsum("sr,cd,rd->sc", np.eye(4) - GAM[mu], U[mu, lex(ym)], u)
        assert np.abs(out[lex(ym)] - e).max() < 1e-14
        # site x = y + mu sees psi(x - mu) = u through the backward hop: (1 + g_mu) U_mu(y)^dag u
        e = np.einsum("sr,dc,rd->sc", np.eye(4) + GAM[mu], U[mu, lex(y)].conj(), u)
        assert np.abs(out[lex(yp)] - e).max() < 1e-14
        nz += 2
    assert np.count_nonzero(np.abs(out).sum(axis=(1, 2)) > 0) == nz


# ---- P12: linearity, translation covariance -------------------------------------------------------

@pytest.mark.parametrize("dims", [(4, 6, 8, 10), (6, 4, 4, 4)])
def test_p12_linearity_and_translation(dims):
    p = oracle.params(dims, KAPPA, mu=0.15, epsilon=0.19, twist_flavor=0)
    U = si.gauge_field(dims, 91, "haar")
    a, b = si.spinor_field(dims, 2, 92), si.spinor_field(dims, 2, 93)
    c = 0.3 - 0.7j
    assert rel(oracle.mat(a + c * b, U, p), oracle.mat(a, U, p) + c * oracle.mat(b, U, p)) < 1e-14
    ref = grid(oracle.mat(a, U, p), dims)
    for mu in range(3):               # spatial shifts commute with M also for antiperiodic time
        ax = AXIS[mu]
        a_s = np.roll(grid(a, dims), 1, axis=ax).reshape(a.shape)
        U_s = np.roll(grid(U, dims), 1, axis=ax).reshape(U.shape)
        assert rel(grid(oracle.mat(a_s, U_s, p), dims), np.roll(ref, 1, axis=ax)) < 1e-15
    pp = oracle.params(dims, KAPPA, mu=0.15, epsilon=0.19, twist_flavor=0, t_boundary=+1)
    ref = grid(oracle.mat(a, U, pp), dims)
    a_s = np.roll(grid(a, dims), 1, axis=1).reshape(a.shape)
    U_s = np.roll(grid(U, dims), 1, axis=1).reshape(U.shape)
    assert rel(grid(oracle.mat(a_s, U_s, pp), dims), np.roll(ref, 1, axis=1)) < 1e-15


# ---- C6: the fused kernels are the compositions PAPER.md:68 names ---------------------------------

@pytest.mark.parametrize("kw", PARAMS)
@pytest.mark.parametrize("parity", [0, 1])
@pytest.mark.parametrize("dag", [0, 1])
def test_fused_kernels_equal_separate_application(kw, parity, dag):
    dims = (4, 6, 4, 4)
    nf = nf_of(kw)
    p = oracle.params(dims, KAPPA, **kw)
    U = si.gauge_field(dims, 101, "haar")
    inp = si.mask_parity(si.spinor_field(dims, nf, 102), dims, 1 - parity)
    x = si.mask_parity(si.spinor_field(dims, nf, 103), dims, parity)
    d = si.mask_parity(oracle.dhop(inp, U, p, dagger=dag), dims, parity)
    k2 = KAPPA * KAPPA
    want = {
        oracle.A: oracle.twist(d, p, 1, dag),
        oracle.A_XPAY: x - k2 * oracle.twist(d, p, 1, dag),
        oracle.B: oracle.twist(x, p, 0, dag) - k2 * d,
        oracle.REC: oracle.twist(x + KAPPA * d, p, 1, dag),
    }
    for kt, w in want.items():
        got = oracle.kernel(inp, x, U, p, parity, dag, kt)
        assert rel(got, w) < 1e-14
        assert np.abs(si.mask_parity(got, dims, 1 - parity)).max() == 0
        # sampled-site entry point agrees with the full one
        sites = si.parity_sites(dims, parity)[::7]
        assert np.array_equal(oracle.kernel_sites(sites, inp, x, U, p, dag, kt), got[:, sites].transpose(1, 0, 2, 3))
    if parity == 0:
        for typ in (oracle.ASYM, oracle.SYM):
            full = oracle.matpc(x, U, p, typ, dagger=dag)
            sites = si.parity_sites(dims, 0)[::5]
            samp = oracle.matpc_sites(sites, x, U, p, typ, dagger=dag)
            assert rel(samp, full[:, sites].transpose(1, 0, 2, 3)) < 1e-14


def test_input_generators_are_special_unitary_and_seeded():
    for kind in ("haar", "near_identity"):
        u = si.gauge_field((2, 2, 2, 2), 7, kind).reshape(-1, 3, 3)
        assert np.abs(u @ u.conj().transpose(0, 2, 1) - np.eye(3)).max() < 1e-14
        assert np.abs(np.linalg.det(u) - 1).max() < 1e-14
        assert np.array_equal(u, si.gauge_field((2, 2, 2, 2), 7, kind).reshape(-1, 3, 3))
    ni = si.gauge_field((2, 2, 2, 2), 7, "near_identity").reshape(-1, 3, 3)
    assert np.abs(ni - np.eye(3)).max() < 1.5                 # near the identity, not Haar
    # Haar first moment vanishes: <U_ij> = 0 ;  second: <|U_ij|^2> = 1/3
    h = si.haar_su3(20000, 3)
    assert np.abs(h.mean(axis=0)).max() < 0.02
    assert np.abs((np.abs(h) ** 2).mean(axis=0) - 1 / 3).max() < 0.01


def test_golden_config1_file_is_what_the_oracle_computes():
    """tests/golden/config1_matpc_asym.txt (written by tests/golden/make_config1_golden.py from oracle/ only) guards the
    oracle's arithmetic against silent changes; it is a regression guard, not a pin (the paper prints no values)."""
    import importlib.util
    import os
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    spec = importlib.util.spec_from_file_location("make_config1_golden", os.path.join(here, "make_config1_golden.py"))
    mk = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mk)
    fields = dict(zip(("matpc_asym", "reconstruct_odd"), mk.compute()))
    n = 0
    for line in open(os.path.join(here, "config1_matpc_asym.txt")):
        if line.startswith("#"):
            continue
        name, s, sp, c, re, im = line.split()
        a = fields[name]
        if int(s) < 0:
            assert abs(np.linalg.norm(a.ravel()) - float(re)) <= 1e-13 * float(re)
        else:
            assert abs(a[0, int(s), int(sp), int(c)] - complex(float(re), float(im))) <= 1e-13
        n += 1
    assert n == 26


def test_p15_chiral_basis_of_the_boundary_is_a_rotation_of_the_declared_basis():
    """include/tm.h TM_BASIS_CHIRAL (reading C12): the chiral matrices written out here satisfy the Clifford
    algebra with gamma5 = g1 g2 g3 g4 = diag(1,1,-1,-1), and S = (1/sqrt2) [[1,1],[1,-1]] maps them onto the oracle's
    non-relativistic matrices: S gamma^chiral S^dag = gamma^nonrel."""
    s = [np.array([[0, 1], [1, 0]], dtype=complex), np.array([[0, -1j], [1j, 0]]), np.array([[1, 0], [0, -1]], dtype=complex)]
    z, one = np.zeros((2, 2), dtype=complex), np.eye(2, dtype=complex)
    gc = [np.block([[z, -1j * sk], [1j * sk, z]]) for sk in s] + [np.block([[z, one], [one, z]])]
    for a in range(4):
        assert np.allclose(gc[a], gc[a].conj().T)
        for b in range(4):
            assert np.allclose(gc[a] @ gc[b] + gc[b] @ gc[a], 2.0 * (a == b) * np.eye(4))
    assert np.allclose(gc[0] @ gc[1] @ gc[2] @ gc[3], np.diag([1, 1, -1, -1]))
    S = np.block([[one, one], [one, -one]]) / np.sqrt(2.0)
    assert np.allclose(S @ S.conj().T, np.eye(4))
    for a in range(4):
        assert np.allclose(S @ gc[a] @ S.conj().T, oracle.gamma(a), atol=1e-15)
    assert np.allclose(S @ np.diag([1, 1, -1, -1]) @ S.conj().T, oracle.gamma(4), atol=1e-15)
