"""Seeded synthetic SU(3) gauge configurations (the ONLY module shared by the oracle-side tests and
the CUDA-side tests).  It holds none of the method's arithmetic: no A_mu, Delta, FFT, p^2, Gram-Schmidt
projection of 1 + i(alpha/2)w, or link transform -- only random numbers and the construction of the
input links that BASELINE.json's ``configs`` prescribe (readings R20, R21).

Random numbers are counter-based (splitmix64 finaliser of ``key + (i+1)*golden``), so value number i
of a stream does not depend on chunking, thread count or generation order.

Array convention: links U have shape (Lt, Lz, Ly, Lx, 4, 3, 3), complex128, site-major, x fastest,
mu = 0..3 = x, y, z, t -- the canonical exchange layout of include/lgf.h.  dims = (Lx, Ly, Lz, Lt).

The paper's own inputs are Monte-Carlo ensembles (Wilson action, beta = 5.8/6.0/6.2, PAPER.md:205-211,
:237) that are not available; these constructions stand in for them with the paper's lattice shapes.
"""
from __future__ import annotations

import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)

# stream ids: independent sub-sequences of one seed
STREAM_H, STREAM_HAAR, STREAM_HOT, STREAM_PHASE = 1, 2, 3, 4


def _mix(z: np.ndarray) -> np.ndarray:
    z = (z ^ (z >> np.uint64(30))) * _M1
    z = (z ^ (z >> np.uint64(27))) * _M2
    return z ^ (z >> np.uint64(31))


def _stream_key(seed: int, stream: int) -> np.uint64:
    with np.errstate(over="ignore"):
        k = _mix(np.array([np.uint64(seed) * _GOLDEN + np.uint64(stream)], dtype=np.uint64))
        return _mix(k ^ np.uint64(0xD6E8FEB86659FD93))[0]


def uniforms(seed: int, stream: int, start: int, count: int) -> np.ndarray:
    """count uniforms in (0, 1): numbers start .. start+count-1 of stream (seed, stream)."""
    with np.errstate(over="ignore"):
        ctr = np.arange(start + 1, start + count + 1, dtype=np.uint64)
        z = _mix(_stream_key(seed, stream) + ctr * _GOLDEN)
    return ((z >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normals(seed: int, stream: int, start: int, count: int) -> np.ndarray:
    """count N(0,1) numbers: normal i = Box-Muller(cos branch) of uniforms 2i, 2i+1."""
    u = uniforms(seed, stream, 2 * start, 2 * count)
    return np.sqrt(-2.0 * np.log(u[0::2])) * np.cos(2.0 * np.pi * u[1::2])


def gell_mann() -> np.ndarray:
    """The eight standard Gell-Mann matrices, tr(l_a l_b) = 2 delta_ab.  Shape (8, 3, 3)."""
    l = np.zeros((8, 3, 3), np.complex128)
    l[0, 0, 1] = l[0, 1, 0] = 1
    l[1, 0, 1], l[1, 1, 0] = -1j, 1j
    l[2, 0, 0], l[2, 1, 1] = 1, -1
    l[3, 0, 2] = l[3, 2, 0] = 1
    l[4, 0, 2], l[4, 2, 0] = -1j, 1j
    l[5, 1, 2] = l[5, 2, 1] = 1
    l[6, 1, 2], l[6, 2, 1] = -1j, 1j
    l[7, 0, 0] = l[7, 1, 1] = 1 / np.sqrt(3.0)
    l[7, 2, 2] = -2 / np.sqrt(3.0)
    return l


def _expi(H: np.ndarray) -> np.ndarray:
    """exp(i H) for stacked hermitian 3x3 H, by scaling (2^-3), Taylor to order 20, and squaring."""
    X = 1j * H / 8.0
    E = np.broadcast_to(np.eye(3, dtype=np.complex128), X.shape).copy()
    T = E.copy()
    for n in range(1, 21):
        T = T @ X / n
        E = E + T
    for _ in range(3):
        E = E @ E
    return E


def haar_su3(seed: int, stream: int, start: int, count: int) -> np.ndarray:
    """count Haar-random SU(3) matrices (numbers start.. of the stream): QR of a complex Ginibre
    matrix, columns rephased by R_ii/|R_ii|, divided by det^(1/3) (R21).  Shape (count, 3, 3)."""
    n = normals(seed, stream, 18 * start, 18 * count).reshape(count, 3, 3, 2)
    Z = (n[..., 0] + 1j * n[..., 1]) / np.sqrt(2.0)
    Q, R = np.linalg.qr(Z)
    d = np.diagonal(R, axis1=-2, axis2=-1)
    Q = Q * (d / np.abs(d))[:, None, :]
    det = np.linalg.det(Q)
    return Q / (det ** (1.0 / 3.0))[:, None, None]


def _site_shape(dims):
    return (dims[3], dims[2], dims[1], dims[0])


def _shift_fwd(h: np.ndarray, mu: int) -> np.ndarray:
    """h(x + mu^) on the (Lt, Lz, Ly, Lx, ...) site grid (periodic)."""
    return np.roll(h, -1, axis=3 - mu)


def smooth_config(dims, eps: float, seed: int, haar: bool = True) -> np.ndarray:
    """U_mu(x) = h(x) exp(i eps H_mu(x)) h(x+mu)^dag, H_mu(x) = sum_a c_a lambda_a with c_a ~ N(0,1)
    (R20), h(x) Haar-random (R21) or the identity (haar=False).  eps = 0 gives a pure-gauge
    configuration h(x) h(x+mu)^dag."""
    dims = tuple(int(v) for v in dims)
    V = dims[0] * dims[1] * dims[2] * dims[3]
    shp = _site_shape(dims)
    if eps != 0.0:
        c = normals(seed, STREAM_H, 0, V * 4 * 8).reshape(V * 4, 8)
        H = np.einsum("na,aij->nij", c.astype(np.complex128), gell_mann())
        E = _expi(eps * H).reshape(shp + (4, 3, 3))
    else:
        E = np.broadcast_to(np.eye(3, dtype=np.complex128), shp + (4, 3, 3)).copy()
    if not haar:
        return np.ascontiguousarray(E)
    h = haar_su3(seed, STREAM_HAAR, 0, V).reshape(shp + (3, 3))
    U = np.empty(shp + (4, 3, 3), np.complex128)
    for mu in range(4):
        hf = _shift_fwd(h, mu)
        U[..., mu, :, :] = h @ E[..., mu, :, :] @ np.conj(np.swapaxes(hf, -1, -2))
    return U


def pure_gauge_config(dims, seed: int) -> np.ndarray:
    """U_mu(x) = h(x) h(x+mu)^dag with Haar h: gauge-equivalent to U = 1 (closed form F -> 1)."""
    return smooth_config(dims, 0.0, seed, haar=True)


def hot_config(dims, seed: int, chunk: int = 1 << 20) -> np.ndarray:
    """Every link an independent Haar-random SU(3) matrix (hot start, config C5)."""
    dims = tuple(int(v) for v in dims)
    V = dims[0] * dims[1] * dims[2] * dims[3]
    U = np.empty((V * 4, 3, 3), np.complex128)
    for s in range(0, V * 4, chunk):
        e = min(s + chunk, V * 4)
        U[s:e] = haar_su3(seed, STREAM_HOT, s, e - s)
    return U.reshape(_site_shape(dims) + (4, 3, 3))


# ---- the same counter-based streams with torch ops (CPU or CUDA) -- for the 64^4 hot start ------------
# The numpy QR above needs minutes for the 67 M links of C5.  These functions draw the SAME uniform and
# normal streams (bit-identical integers; log / cos may differ from numpy's in the last ulp) and
# orthonormalise the Ginibre matrix by classical Gram-Schmidt on its columns, which is the QR factor with a
# positive diagonal, i.e. the same Haar recipe (R21).  Still no method arithmetic: input construction only.
def _torch_uniforms(torch, seed: int, stream: int, start: int, count: int, device):
    key = int(_stream_key(seed, stream))
    key = key - (1 << 64) if key >= (1 << 63) else key
    golden = int(_GOLDEN) - (1 << 64)
    m1, m2 = int(_M1) - (1 << 64), int(_M2) - (1 << 64)

    def lsr(z, k):                                    # logical shift right of an int64 bit pattern
        return (z >> k) & ((1 << (64 - k)) - 1)

    ctr = torch.arange(start + 1, start + count + 1, dtype=torch.int64, device=device)
    z = key + ctr * golden
    z = (z ^ lsr(z, 30)) * m1
    z = (z ^ lsr(z, 27)) * m2
    z = z ^ lsr(z, 31)
    return (lsr(z, 11).to(torch.float64) + 0.5) * (1.0 / 9007199254740992.0)


def _torch_normals(torch, seed: int, stream: int, start: int, count: int, device):
    u = _torch_uniforms(torch, seed, stream, 2 * start, 2 * count, device)
    return torch.sqrt(-2.0 * torch.log(u[0::2])) * torch.cos(2.0 * np.pi * u[1::2])


def haar_su3_torch(seed: int, stream: int, start: int, count: int, device="cpu"):
    """count Haar-random SU(3) matrices as a torch complex128 tensor (count, 3, 3) on `device`."""
    import torch

    n = _torch_normals(torch, seed, stream, 18 * start, 18 * count, device).reshape(count, 3, 3, 2)
    Z = torch.complex(n[..., 0], n[..., 1]) / np.sqrt(2.0)
    cols = []
    for j in range(3):                                # Gram-Schmidt on columns = Q of QR with R_jj > 0
        v = Z[:, :, j]
        for _ in range(2):                            # orthogonalise twice: unitary to rounding
            for q in cols:
                v = v - q * (q.conj() * v).sum(dim=1, keepdim=True)
        cols.append(v / torch.linalg.vector_norm(v, dim=1, keepdim=True))
    Q = torch.stack(cols, dim=2)
    det = torch.linalg.det(Q)
    return Q / (det ** (1.0 / 3.0))[:, None, None]


def hot_config_torch(dims, seed: int, device="cpu", chunk: int = 1 << 22):
    """hot_config with torch ops: every link Haar-random; returns a torch complex128 tensor of shape
    (Lt, Lz, Ly, Lx, 4, 3, 3) on `device`.  Same streams as hot_config, Gram-Schmidt instead of LAPACK QR."""
    import torch

    dims = tuple(int(v) for v in dims)
    V = dims[0] * dims[1] * dims[2] * dims[3]
    U = torch.empty((V * 4, 3, 3), dtype=torch.complex128, device=device)
    for s in range(0, V * 4, chunk):
        e = min(s + chunk, V * 4)
        U[s:e] = haar_su3_torch(seed, STREAM_HOT, s, e - s, device)
    return U.reshape(_site_shape(dims) + (4, 3, 3))


def abelian_config(dims, amp: float, seed: int) -> np.ndarray:
    """Diagonal links U = diag(e^{i p1}, e^{i p2}, e^{-i(p1+p2)}) with phases p ~ amp * N(0,1):
    a small-field abelian configuration on which the linearised iteration is exactly solvable."""
    dims = tuple(int(v) for v in dims)
    V = dims[0] * dims[1] * dims[2] * dims[3]
    p = amp * normals(seed, STREAM_PHASE, 0, V * 4 * 2).reshape(V * 4, 2)
    U = np.zeros((V * 4, 3, 3), np.complex128)
    U[:, 0, 0] = np.exp(1j * p[:, 0])
    U[:, 1, 1] = np.exp(1j * p[:, 1])
    U[:, 2, 2] = np.exp(-1j * (p[:, 0] + p[:, 1]))
    return U.reshape(_site_shape(dims) + (4, 3, 3))


# BASELINE.json `configs`, seeds as proposed in SURVEY.md section 8(d)
CONFIGS = {
    "C1": dict(dims=(8, 8, 8, 8), kind="smooth", eps=0.2, seed=1001, alpha=0.08),
    "C2": dict(dims=(16, 16, 16, 16), kind="smooth", eps=0.2, seed=1002, alpha=0.08),
    "C2pg": dict(dims=(16, 16, 16, 16), kind="smooth", eps=0.0, seed=1003, alpha=0.08),
    "C3": dict(dims=(32, 32, 32, 32), kind="smooth", eps=0.3, seed=1004, alpha=0.08),
    "C4": dict(dims=(24, 24, 24, 48), kind="smooth", eps=0.3, seed=1005, alpha=0.08),
    "C5": dict(dims=(64, 64, 64, 64), kind="hot", eps=None, seed=1006, alpha=0.08),
}


def make_config(name: str, seed_offset: int = 0) -> np.ndarray:
    """Build the named BASELINE.json configuration (seed_offset selects another ensemble member)."""
    c = CONFIGS[name]
    seed = c["seed"] + 7919 * int(seed_offset)
    if c["kind"] == "hot":
        return hot_config(c["dims"], seed)
    return smooth_config(c["dims"], c["eps"], seed, haar=True)
