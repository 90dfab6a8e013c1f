"""ctypes front end of the CPU oracle (oracle/tm_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It shares no code with paper_1311_4462_b200 (the CUDA path) and never imports it.

Arrays are numpy complex128, C-contiguous:
    spinor : [nf, V, 4, 3]   (nf = 1 degenerate, 2 doublet), lex = x1 + X (x2 + Y (x3 + Z x4))
    gauge  : [4, V, 3, 3]    U_mu(x), link from x to x + mu_hat
Operator definitions and the paper passages they follow are in the header of tm_oracle.c.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tm_oracle.c")
_LIB = os.path.join(_HERE, "libtm_oracle.so")

A, A_XPAY, B, REC = 0, 1, 2, 3
ASYM, SYM = 0, 1
EVEN, ODD = 0, 1


def build(force=False):
    """Compile tm_oracle.c with gcc (also called by __graft_entry__.build())."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fcx-limited-range", "-Wall", "-Wextra",
               "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class Params(ctypes.Structure):
    _fields_ = [("X", ctypes.c_int * 4), ("kappa", ctypes.c_double), ("mu", ctypes.c_double),
                ("epsilon", ctypes.c_double), ("twist_flavor", ctypes.c_int),
                ("t_boundary", ctypes.c_int)]


def params(dims, kappa, mu, epsilon=0.0, twist_flavor=1, t_boundary=-1):
    p = Params()
    p.X[:] = [int(d) for d in dims]
    p.kappa, p.mu, p.epsilon = float(kappa), float(mu), float(epsilon)
    p.twist_flavor, p.t_boundary = int(twist_flavor), int(t_boundary)
    return p


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        dp = ctypes.c_void_p
        pp = ctypes.POINTER(Params)
        i, l = ctypes.c_int, ctypes.c_long
        _lib.tmo_num_threads.restype = i
        _lib.tmo_set_num_threads.argtypes = [i]
        _lib.tmo_gamma.argtypes = [i, dp]
        _lib.tmo_site_parity.argtypes = [l, ctypes.POINTER(i)]
        _lib.tmo_dhop.argtypes = [dp, dp, dp, pp, i]
        _lib.tmo_twist.argtypes = [dp, dp, pp, i, i]
        _lib.tmo_mat.argtypes = [dp, dp, dp, pp, i]
        _lib.tmo_kernel.argtypes = [dp, dp, dp, dp, pp, i, i, i]
        _lib.tmo_kernel_sites.argtypes = [dp, dp, l, dp, dp, dp, pp, i, i]
        _lib.tmo_matpc.argtypes = [dp, dp, dp, pp, i, i]
        _lib.tmo_reconstruct_odd.argtypes = [dp, dp, dp, dp, pp]
        _lib.tmo_matpc_sites.argtypes = [dp, dp, l, dp, dp, pp, i, i]
    return _lib


def num_threads():
    return lib().tmo_num_threads()


def set_num_threads(n):
    lib().tmo_set_num_threads(int(n))


def _nf(p):
    return 2 if p.twist_flavor == 0 else 1


def _vol(p):
    return int(p.X[0]) * int(p.X[1]) * int(p.X[2]) * int(p.X[3])


def _spinor(a, p, name):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    if a.shape != (_nf(p), _vol(p), 4, 3):
        raise ValueError(f"{name}: shape {a.shape}, expected {(_nf(p), _vol(p), 4, 3)}")
    return a


def _gauge(g, p):
    g = np.ascontiguousarray(g, dtype=np.complex128)
    if g.shape != (4, _vol(p), 3, 3):
        raise ValueError(f"gauge: shape {g.shape}, expected {(4, _vol(p), 3, 3)}")
    return g


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _check(err, what):
    if err:
        raise RuntimeError(f"oracle {what} failed with code {err}")


def gamma(idx):
    """gamma_1..gamma_4 for idx 0..3, gamma_5 (as the product) for idx 4; 4x4 complex."""
    out = np.zeros((4, 4), dtype=np.complex128)
    lib().tmo_gamma(int(idx), _ptr(out))
    return out


def site_parity(dims):
    """Parity (x1+x2+x3+x4) mod 2 of every lexicographic site, int array [V]."""
    X, Y, Z, T = (int(d) for d in dims)
    x = np.arange(X).reshape(1, 1, 1, X)
    y = np.arange(Y).reshape(1, 1, Y, 1)
    z = np.arange(Z).reshape(1, Z, 1, 1)
    t = np.arange(T).reshape(T, 1, 1, 1)
    return ((x + y + z + t) & 1).reshape(-1)


def dhop(psi, gauge, p, dagger=0):
    psi, gauge = _spinor(psi, p, "psi"), _gauge(gauge, p)
    out = np.zeros_like(psi)
    _check(lib().tmo_dhop(_ptr(out), _ptr(psi), _ptr(gauge), ctypes.byref(p), int(dagger)), "dhop")
    return out


def twist(psi, p, inverse=0, dagger=0):
    psi = _spinor(psi, p, "psi")
    out = np.zeros_like(psi)
    _check(lib().tmo_twist(_ptr(out), _ptr(psi), ctypes.byref(p), int(inverse), int(dagger)), "twist")
    return out


def mat(psi, gauge, p, dagger=0):
    """M psi = (R - kappa D_hop) psi on the full lattice."""
    psi, gauge = _spinor(psi, p, "psi"), _gauge(gauge, p)
    out = np.zeros_like(psi)
    _check(lib().tmo_mat(_ptr(out), _ptr(psi), _ptr(gauge), ctypes.byref(p), int(dagger)), "mat")
    return out


def kernel(inp, x, gauge, p, parity, dagger, kernel_type):
    """One fused kernel (A / A_XPAY / B / REC); full-lattice arrays, result nonzero on `parity` only."""
    inp, gauge = _spinor(inp, p, "in"), _gauge(gauge, p)
    x = None if x is None else _spinor(x, p, "x")
    out = np.zeros_like(inp)
    _check(lib().tmo_kernel(_ptr(out), _ptr(inp), _ptr(x), _ptr(gauge), ctypes.byref(p), int(parity),
                            int(dagger), int(kernel_type)), "kernel")
    return out


def kernel_sites(sites, inp, x, gauge, p, dagger, kernel_type):
    """The same kernel at the listed lexicographic output sites only -> [n, nf, 4, 3]."""
    inp, gauge = _spinor(inp, p, "in"), _gauge(gauge, p)
    x = None if x is None else _spinor(x, p, "x")
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.zeros((len(sites), _nf(p), 4, 3), dtype=np.complex128)
    _check(lib().tmo_kernel_sites(_ptr(out), _ptr(sites), len(sites), _ptr(inp), _ptr(x), _ptr(gauge),
                                  ctypes.byref(p), int(dagger), int(kernel_type)), "kernel_sites")
    return out


def matpc(inp, gauge, p, matpc_type, dagger=0):
    """LHS of Eq. (2.2) (ASYM) or Eq. (2.3) (SYM) on the even sites of a full-lattice array."""
    inp, gauge = _spinor(inp, p, "in"), _gauge(gauge, p)
    out = np.zeros_like(inp)
    _check(lib().tmo_matpc(_ptr(out), _ptr(inp), _ptr(gauge), ctypes.byref(p), int(matpc_type),
                           int(dagger)), "matpc")
    return out


def matpc_sites(sites, inp, gauge, p, matpc_type, dagger=0):
    inp, gauge = _spinor(inp, p, "in"), _gauge(gauge, p)
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.zeros((len(sites), _nf(p), 4, 3), dtype=np.complex128)
    _check(lib().tmo_matpc_sites(_ptr(out), _ptr(sites), len(sites), _ptr(inp), _ptr(gauge),
                                 ctypes.byref(p), int(matpc_type), int(dagger)), "matpc_sites")
    return out


def reconstruct_odd(psi_e, b_o, gauge, p):
    """Eq. (2.4): psi_o = R_oo^{-1} (b_o + kappa D_oe psi_e); result nonzero on odd sites only."""
    psi_e, b_o, gauge = _spinor(psi_e, p, "psi_e"), _spinor(b_o, p, "b_o"), _gauge(gauge, p)
    out = np.zeros_like(psi_e)
    _check(lib().tmo_reconstruct_odd(_ptr(out), _ptr(psi_e), _ptr(b_o), _ptr(gauge), ctypes.byref(p)),
           "reconstruct_odd")
    return out


# ---- compositions of the primitives above (plain definitions; no new arithmetic) ---------------------------

def _mask(a, p, parity):
    """Zero the sites of the other parity (full-lattice array in, full-lattice array out)."""
    par = site_parity([p.X[k] for k in range(4)])
    out = np.array(a, dtype=np.complex128, copy=True)
    out[:, par != parity] = 0
    return out


def hop_xpay(inp, x, gauge, p, parity, dagger, coeff):
    """out_p = x_p + coeff (D_hop in)_p  with no twist: the plain forms the product exposes as TM_DSLASH_XPAY
    (coeff = -kappa^2) and TM_DSLASH_AXPY (coeff = +kappa)."""
    return _mask(x, p, parity) + coeff * _mask(dhop(inp, gauge, p, dagger), p, parity)


def kernel_twist_in(inp, x, gauge, p, parity, dagger, form):
    """The fused "D R^-1" forms (the inverse twist acts on the INPUT field, then the hopping term):
    form "A": R^-1 D_hop R^-1 in;  "REC": R^-1 (x + kappa D_hop R^-1 in);  "AXPY": x + kappa D_hop R^-1 in,
    restricted to `parity`; dagger: R -> R^dag, D_hop -> D_hop^dag.  Compositions of twist, kernel and hop_xpay."""
    t = twist(_mask(inp, p, 1 - parity), p, 1, dagger)
    if form == "A":
        return kernel(t, None, gauge, p, parity, dagger, A)
    if form == "REC":
        return kernel(t, x, gauge, p, parity, dagger, REC)
    if form == "AXPY":
        return hop_xpay(t, x, gauge, p, parity, dagger, p.kappa)
    raise ValueError(form)


def matpc_adjoint(inp, gauge, p, matpc_type):
    """The adjoint of the even-even operators written out from D_hop^dag and R^dag (C7):
    ASYM: (R_ee^dag - kappa^2 D_eo^dag R_oo^dag^-1 D_oe^dag) in_e
    SYM : (1 - kappa^2 D_eo^dag R_oo^dag^-1 D_oe^dag R_ee^dag^-1) in_e        (adjoint taken term by term)."""
    in_e = _mask(inp, p, EVEN)
    k2 = p.kappa * p.kappa
    if matpc_type == ASYM:
        t_o = twist(_mask(dhop(in_e, gauge, p, 1), p, ODD), p, 1, 1)
        return twist(in_e, p, 0, 1) - k2 * _mask(dhop(t_o, gauge, p, 1), p, EVEN)
    y_e = twist(in_e, p, 1, 1)
    t_o = twist(_mask(dhop(y_e, gauge, p, 1), p, ODD), p, 1, 1)
    return in_e - k2 * _mask(dhop(t_o, gauge, p, 1), p, EVEN)


def prepare_rhs(b, gauge, p, matpc_type):
    """Right-hand side of Eq. (2.2) / (2.3) in the reading C4: b_e + kappa D_eo R_oo^-1 b_o, times R_ee^-1 for SYM."""
    t_o = twist(_mask(b, p, ODD), p, 1, 0)
    r = _mask(b, p, EVEN) + p.kappa * _mask(dhop(t_o, gauge, p, 0), p, EVEN)
    return r if matpc_type == ASYM else twist(r, p, 1, 0)
