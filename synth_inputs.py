"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no gamma matrices, no hopping term, no twist):
it only draws random SU(3) links and Gaussian spinors in the host canonical order, and does the
pure index bookkeeping between full-lattice lexicographic arrays and single-parity ("checkerboard")
arrays.  Neither oracle/ nor paper_1311_4462_b200/ imports it; callers pass its arrays to both.

The lattices stand in for the gauge ensembles behind PAPER.md:95-134 (not available offline); the
recipes are BASELINE.json's configs (DESIGN.md section "Input recipe"):
  * Haar-random SU(3): Gram-Schmidt (= QR with the diagonal of R made real positive) of a complex
    Gaussian 3x3, divided by det^(1/3);
  * near-identity SU(3): exp(i * 0.3 * H), H traceless Hermitian Gaussian;
  * spinors: re and im iid N(0, 1).
Random numbers come from numpy's counter-based Philox generator keyed by (seed, stream).
"""
import numpy as np

STREAM_GAUGE, STREAM_SPINOR = 1, 2


def _rng(seed, stream):
    return np.random.Generator(np.random.Philox(key=[int(seed), int(stream)]))


def volume(dims):
    X, Y, Z, T = (int(d) for d in dims)
    return X * Y * Z * T


def _cgauss(rng, shape):
    out = np.empty(shape, dtype=np.complex128)
    out.real = rng.standard_normal(shape)
    out.imag = rng.standard_normal(shape)
    return out


def haar_su3(n, seed, stream=STREAM_GAUGE, chunk=1 << 20):
    """n Haar-distributed SU(3) matrices, [n, 3, 3] complex128."""
    rng = _rng(seed, stream)
    out = np.empty((n, 3, 3), dtype=np.complex128)
    for lo in range(0, n, chunk):
        hi = min(n, lo + chunk)
        a = _cgauss(rng, (hi - lo, 3, 3))
        q = np.empty_like(a)
        for j in range(3):                       # Gram-Schmidt on the columns
            v = a[:, :, j].copy()
            for k in range(j):
                v -= np.sum(q[:, :, k].conj() * v, axis=1, keepdims=True) * q[:, :, k]
            q[:, :, j] = v / np.linalg.norm(v, axis=1, keepdims=True)
        det = np.linalg.det(q)
        out[lo:hi] = q / np.exp(1j * np.angle(det) / 3.0)[:, None, None]
    return out


def near_identity_su3(n, seed, scale=0.3, stream=STREAM_GAUGE, chunk=1 << 20):
    """n matrices exp(i * scale * H), H traceless Hermitian Gaussian, [n, 3, 3] complex128."""
    rng = _rng(seed, stream)
    out = np.empty((n, 3, 3), dtype=np.complex128)
    for lo in range(0, n, chunk):
        hi = min(n, lo + chunk)
        m = hi - lo
        h = np.zeros((m, 3, 3), dtype=np.complex128)
        d = rng.standard_normal((m, 3))
        d -= d.mean(axis=1, keepdims=True)
        for j in range(3):
            h[:, j, j] = d[:, j]
        for j in range(3):
            for k in range(j + 1, 3):
                z = (rng.standard_normal(m) + 1j * rng.standard_normal(m)) / np.sqrt(2.0)
                h[:, j, k] = z
                h[:, k, j] = z.conj()
        w, v = np.linalg.eigh(h)                 # exp(i s H) = V diag(exp(i s w)) V^dagger
        out[lo:hi] = (v * np.exp(1j * scale * w)[:, None, :]) @ v.conj().transpose(0, 2, 1)
    return out


def gauge_field(dims, seed, kind="haar"):
    """Host canonical gauge field [4, V, 3, 3] (mu, lexicographic site, row, col)."""
    V = volume(dims)
    if kind == "haar":
        u = haar_su3(4 * V, seed)
    elif kind == "near_identity":
        u = near_identity_su3(4 * V, seed)
    elif kind == "unit":
        u = np.broadcast_to(np.eye(3, dtype=np.complex128), (4 * V, 3, 3)).copy()
    else:
        raise ValueError(kind)
    return u.reshape(4, V, 3, 3)


def spinor_field(dims, nf, seed, stream=STREAM_SPINOR):
    """Host canonical full-lattice spinor [nf, V, 4, 3], re and im iid N(0,1)."""
    return _cgauss(_rng(seed, stream), (nf, volume(dims), 4, 3))


# ---- pure index bookkeeping: full lattice <-> single parity --------------------------------

def parity_sites(dims, parity):
    """Lexicographic indices of the sites of one parity, ordered by checkerboard index i = lex // 2."""
    X, Y, Z, T = (int(d) for d in dims)
    x = np.arange(X).reshape(1, 1, 1, X)
    y = np.arange(Y).reshape(1, 1, Y, 1)
    z = np.arange(Z).reshape(1, Z, 1, 1)
    t = np.arange(T).reshape(T, 1, 1, 1)
    par = ((x + y + z + t) & 1).reshape(-1)
    return np.nonzero(par == int(parity))[0]


def to_parity(full, dims, parity):
    """[nf, V, 4, 3] -> [nf, V/2, 4, 3]: the sites of `parity` in checkerboard order."""
    return np.ascontiguousarray(full[:, parity_sites(dims, parity)])


def from_parity(cb, dims, parity, out=None):
    """Scatter a single-parity array back into a (zero-initialised or given) full-lattice array."""
    nf = cb.shape[0]
    if out is None:
        out = np.zeros((nf, volume(dims), 4, 3), dtype=cb.dtype)
    out[:, parity_sites(dims, parity)] = cb
    return out


def mask_parity(full, dims, parity):
    """Copy of `full` with the sites of the other parity set to zero."""
    out = np.zeros_like(full)
    idx = parity_sites(dims, parity)
    out[:, idx] = full[:, idx]
    return out
