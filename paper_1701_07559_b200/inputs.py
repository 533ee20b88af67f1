"""Seeded synthetic inputs shared (as DATA) by the oracle and the CUDA path.

This module holds none of the method's arithmetic: no gamma matrices, no hopping term, no
fifth-dimension operator.  It only draws random numbers and exponentiates Hermitian 3x3
matrices, i.e. it makes the gauge field and the sources that both sides are then handed.

Recipe:
  links   U_mu(x) = exp(i eps H), H = (G + G^+)/2 - tr/3, G_ij = N(0,1) + i N(0,1) i.i.d.
          These stand in for the paper's gradient-flowed MILC HISQ configurations
          (Table I), which are not available offline.
  source  Gaussian complex on every (x,s,spin,colour), re, im ~ N(0,1), not normalised;
          or a point source at the origin on the two domain walls.
  RNG     counter-based: value = f(seed, field id, element index), so the result does not
          depend on generation order or device (up to the last bit of log/cos).
Layouts are the canonical interchange layouts of include/mdwf.h.
"""
import math

import torch

_MASK64 = (1 << 64) - 1


def _to_i64(v: int) -> int:
    v &= _MASK64
    return v - (1 << 64) if v >= (1 << 63) else v


_C1 = _to_i64(0x9E3779B97F4A7C15)
_C2 = _to_i64(0xBF58476D1CE4E5B9)
_C3 = _to_i64(0x94D049BB133111EB)


def _lsr(x: torch.Tensor, k: int) -> torch.Tensor:
    """logical shift right on int64 tensors"""
    return (x >> k) & ((1 << (64 - k)) - 1)


def _mix(z: torch.Tensor) -> torch.Tensor:
    """splitmix64 finaliser (wrapping int64 arithmetic)."""
    z = (z ^ _lsr(z, 30)) * _C2
    z = (z ^ _lsr(z, 27)) * _C3
    return z ^ _lsr(z, 31)


def _uniform(seed: int, field: int, n: int, stream: int, device) -> torch.Tensor:
    """n uniforms in (0,1), element i of stream `stream` of field `field`."""
    idx = torch.arange(n, dtype=torch.int64, device=device)
    key = _to_i64((seed * 0x100000001B3 + field * 0x1000193 + stream * 0x9E3779B1 + 0x1234567) & _MASK64)
    z = _mix(_mix(idx * _C1 + key) + key)
    return (_lsr(z, 11).to(torch.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normal(seed: int, field: int, n: int, device="cpu") -> torch.Tensor:
    """n standard normals (Box-Muller on two counter-based uniform streams), float64."""
    u1 = _uniform(seed, field, n, 0, device)
    u2 = _uniform(seed, field, n, 1, device)
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2)


def complex_normal(seed: int, field: int, n: int, device="cpu") -> torch.Tensor:
    return torch.complex(normal(seed, 2 * field, n, device), normal(seed, 2 * field + 1, n, device))


def traceless_hermitian(seed: int, field: int, n: int, device="cpu") -> torch.Tensor:
    """n random traceless Hermitian 3x3 matrices H = (G + G^+)/2 - tr/3."""
    G = complex_normal(seed, field, n * 9, device).reshape(n, 3, 3)
    H = 0.5 * (G + G.conj().transpose(-1, -2))
    tr = torch.diagonal(H, dim1=-2, dim2=-1).sum(-1).real / 3.0
    eye = torch.eye(3, dtype=H.dtype, device=device)
    return H - tr[:, None, None] * eye


def su3_exp(H: torch.Tensor, eps: float) -> torch.Tensor:
    """exp(i eps H) for a batch of Hermitian traceless H (complex128)."""
    out = torch.empty_like(H)
    chunk = 1 << 20
    for i in range(0, H.shape[0], chunk):
        out[i:i + chunk] = torch.linalg.matrix_exp((1j * eps) * H[i:i + chunk])
    return out


def gauge_field(L, eps: float, seed: int, device="cpu") -> torch.Tensor:
    """U[t][z][y][x][mu][row][col] complex128, U = exp(i eps H); eps = 0 gives unit links."""
    Lx, Ly, Lz, Lt = L
    n = Lx * Ly * Lz * Lt * 4
    H = traceless_hermitian(seed, 1, n, device)
    U = su3_exp(H, eps)
    return U.reshape(Lt, Lz, Ly, Lx, 4, 3, 3).contiguous()


def gaussian_source(L, L5: int, seed: int, device="cpu") -> torch.Tensor:
    """psi[s][t][z][y][x][spin][colour] complex128, re, im ~ N(0,1)."""
    Lx, Ly, Lz, Lt = L
    n = L5 * Lt * Lz * Ly * Lx * 12
    return complex_normal(seed + 1000, 7, n, device).reshape(L5, Lt, Lz, Ly, Lx, 4, 3).contiguous()


def point_source(L, L5: int, spin: int, colour: int, device="cpu") -> torch.Tensor:
    """delta at the 4D origin on the walls: upper spins (P+) on s = 0, lower spins (P-) on s = L5-1
    (the wall injection without the Moebius D_- factor)."""
    Lx, Ly, Lz, Lt = L
    b = torch.zeros(L5, Lt, Lz, Ly, Lx, 4, 3, dtype=torch.complex128, device=device)
    s = 0 if spin < 2 else L5 - 1
    b[s, 0, 0, 0, 0, spin, colour] = 1.0
    return b


def random_su3(seed: int, n: int, device="cpu") -> torch.Tensor:
    """n Haar-ish SU(3) matrices (exp(i H) with O(1) H) -- gauge transformations for tests."""
    return su3_exp(traceless_hermitian(seed, 3, n, device), 1.0)


# The five workloads of BASELINE.json `configs` (index 0..4 = configs 1..5 of SURVEY.md 8(d)).
CONFIGS = [
    dict(name="4^4xL5=8", L=(4, 4, 4, 4), L5=8, M5=1.3, b5=1.5, c5=0.5, mf=0.05, eps=0.3, seed=0,
         source="gaussian", ladder="d", reconstruct=18),
    dict(name="16^3x48xL5=12", L=(16, 16, 16, 48), L5=12, M5=1.3, b5=1.75, c5=0.75, mf=0.02, eps=0.2, seed=1,
         source="gaussian", ladder="ds", reconstruct=18),
    dict(name="24^3x64xL5=8", L=(24, 24, 24, 64), L5=8, M5=1.2, b5=1.25, c5=0.25, mf=0.01, eps=0.15, seed=2,
         source="point12", ladder="ds", reconstruct=18),
    dict(name="32^3x96xL5=12", L=(32, 32, 32, 96), L5=12, M5=1.1, b5=1.5, c5=0.5, mf=0.005, eps=0.1, seed=3,
         source="gaussian", ladder="dsh", reconstruct=12),
    dict(name="48^3x96xL5=12", L=(48, 48, 48, 96), L5=12, M5=1.1, b5=1.5, c5=0.5, mf=0.002, eps=0.1, seed=4,
         source="gaussian", ladder="dh", reconstruct=18),
]
