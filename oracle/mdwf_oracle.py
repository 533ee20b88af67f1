"""CPU oracle for the MDWF even-odd operator and its CG solve.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It never imports paper_1701_07559_b200 (the CUDA path) and the CUDA
path never imports it.

The primitives (hopping term D3, Lambda D5, A^{-1} D6) are the plain C loops of
oracle/mdwf_oracle.c; this file composes them *step by step* in the order of SURVEY.md
section 8(c) D6-D9:

  D6  D      = A - (1/2) H B,   A = alpha + beta Lambda,   B = b5 + c5 Lambda
      (this is D_W (b5 + c5 Lambda) + (1 - Lambda) with D_W = (4 - M5) - H/2 the Wilson kernel of
       Eq. (2))
  D7  Mpc    = A - (1/4) H_oe B A^{-1} H_eo B          on odd sites ("asymmetric")
      Mpc^+  = A^+ - (1/4) B^+ H'_oe A^{-+} B^+ H'_eo   with H' = gamma5 H gamma5 = H^+
  D8  Schur: b'_o = b_o - D_oe A^{-1} b_e ; Mpc x_o = b'_o ; x_e = A^{-1}(b_e - D_eo x_o)
  D9  CGLS on Mpc^+ Mpc.

All vectors are full-lattice complex128 arrays psi[s][t][z][y][x][spin][colour]; a
single-parity vector is such an array that vanishes on the other parity.  Every step works
on an explicit list of 4D sites, so the same code evaluates the operator on the whole
lattice or on a handful of sampled sites (Mpc_at_sites).

Flop convention (D10), used wherever a rate is quoted: F_Mpc(L5) = 2880 + 48 L5 per odd
5D site per application of Mpc or Mpc^+.

SURVEY.md 8(f) rows, at the end of the class (each with its own pin in tests/test_oracle_pins3.py):
  NEXT-1  Mpc_sym = 1 - (1/4) A^{-1} H_oe B A^{-1} H_eo B = A^{-1} Mpc, its adjoint and the solve through it
          ("symmetric" preconditioning)
  NEXT-3  4D <-> 5D maps around the solve (Eq. (5)): wall source and D_- lift of a 4D source,
          wall projection q = P- psi_0 + P+ psi_{L5-1}, midpoint field

Pins: tests/test_oracle_pins.py (P1-P9 of SURVEY.md 8(c)).  Unpinned: nothing in this file;
the mixed-precision ladder lives only in the CUDA path and is "parity unpinned" beyond the
true residual.
"""
import ctypes
import os

import numpy as np

from . import build as _build

_lib = None


def _load():
    global _lib
    if _lib is None:
        path = _build.build()
        lib = ctypes.CDLL(path)
        P = ctypes.c_void_p
        I64 = ctypes.c_int64
        D = ctypes.c_double
        lib.orc_gamma.argtypes = [ctypes.c_int, P]
        lib.orc_num_threads.restype = ctypes.c_int
        lib.orc_hop.argtypes = [P, ctypes.c_int, P, P, P, P, I64, ctypes.c_int]
        lib.orc_s_affine.argtypes = [I64, ctypes.c_int, D, D, D, P, P, P, I64, ctypes.c_int]
        lib.orc_Ainv_table.argtypes = [ctypes.c_int, D, D, D, P]
        lib.orc_Ainv.argtypes = [I64, ctypes.c_int, D, D, D, P, P, P, I64, ctypes.c_int]
        lib.orc_axpby.argtypes = [I64, ctypes.c_int, D, P, D, P, P, P, I64]
        lib.orc_redot.argtypes = [I64, ctypes.c_int, P, P, P, I64]
        lib.orc_redot.restype = D
        _lib = lib
    return _lib


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def num_threads():
    return int(_load().orc_num_threads())


def flops_per_site(L5):
    """D10: fixed flop count per odd 5D site per Mpc (or Mpc^+) application."""
    return 2880 + 48 * L5


def gamma(mu):
    """gamma_mu (mu = 0..3 for x,y,z,t; 4 for gamma_5) in the DeGrand-Rossi basis (D2)."""
    buf = np.zeros(32)
    _load().orc_gamma(mu, _p(buf))
    return (buf[0::2] + 1j * buf[1::2]).reshape(4, 4)


def Ainv_plus_table(L5, alpha, beta, mf):
    """Closed form (D6) of the P+ block of A^{-1}; the P- block is its transpose."""
    t = np.zeros((L5, L5))
    _load().orc_Ainv_table(L5, alpha, beta, mf, _p(t))
    return t


class MdwfOracle:
    def __init__(self, L, L5, M5, b5, c5, mf, U):
        """L = (Lx, Ly, Lz, Lt); U complex128 [Lt][Lz][Ly][Lx][mu][row][col] (plain SU(3) links)."""
        self.L = tuple(int(v) for v in L)
        assert all(v % 2 == 0 for v in self.L), "all extents must be even (D1)"
        self.L5 = int(L5)
        self.M5, self.b5, self.c5, self.mf = float(M5), float(b5), float(c5), float(mf)
        self.alpha = self.b5 * (4.0 - self.M5) + 1.0
        self.beta = self.c5 * (4.0 - self.M5) - 1.0
        Lx, Ly, Lz, Lt = self.L
        self.V4 = Lx * Ly * Lz * Lt
        self.shape = (self.L5, Lt, Lz, Ly, Lx, 4, 3)
        self.U = np.ascontiguousarray(U, dtype=np.complex128)
        assert self.U.shape == (Lt, Lz, Ly, Lx, 4, 3, 3)
        self._Lc = (ctypes.c_int * 4)(*self.L)
        idx = np.arange(self.V4, dtype=np.int64)
        x = idx % Lx
        y = (idx // Lx) % Ly
        z = (idx // (Lx * Ly)) % Lz
        t = idx // (Lx * Ly * Lz)
        par = (x + y + z + t) & 1
        self.sites_even = np.ascontiguousarray(idx[par == 0])
        self.sites_odd = np.ascontiguousarray(idx[par == 1])
        self.sites_all = idx
        self.lib = _load()

    # ---- bookkeeping -----------------------------------------------------------------
    def zeros(self):
        return np.zeros(self.shape, dtype=np.complex128)

    def sites(self, parity):
        return (self.sites_even, self.sites_odd, self.sites_all)[parity]

    def neighbours(self, sites):
        """4D lexicographic indices of the 8 nearest neighbours of the given sites (unique, sorted)."""
        Lx, Ly, Lz, Lt = self.L
        s = np.asarray(sites, dtype=np.int64)
        c = [s % Lx, (s // Lx) % Ly, (s // (Lx * Ly)) % Lz, s // (Lx * Ly * Lz)]
        out = []
        for mu in range(4):
            for d in (+1, -1):
                cc = [v.copy() for v in c]
                cc[mu] = (cc[mu] + d) % self.L[mu]
                out.append(cc[0] + Lx * (cc[1] + Ly * (cc[2] + Lz * cc[3])))
        return np.unique(np.concatenate(out)).astype(np.int64)

    def pack_parity(self, v, parity):
        """full [s][t][z][y][x][4][3] -> single-parity [s][cb][4][3], cb = lex/2 over sites of that parity."""
        flat = v.reshape(self.L5, self.V4, 4, 3)
        return np.ascontiguousarray(flat[:, self.sites(parity)])

    def unpack_parity(self, vp, parity):
        out = self.zeros()
        out.reshape(self.L5, self.V4, 4, 3)[:, self.sites(parity)] = vp
        return out

    # ---- primitives on site lists ----------------------------------------------------
    def hop(self, v, sites, dagger=False, out=None):
        """D3 on the listed sites: out(x,s) = sum_mu (1 -+ gamma_mu) U psi(x+mu) + (1 +- gamma_mu) U^+ psi(x-mu)."""
        out = self.zeros() if out is None else out
        sites = np.ascontiguousarray(sites, dtype=np.int64)
        self.lib.orc_hop(self._Lc, self.L5, _p(self.U), _p(v), _p(out), _p(sites), len(sites), int(dagger))
        return out

    def s_affine(self, a, b, v, sites, dagger=False, out=None):
        """out = a v + b Lambda v (D5) on the listed sites."""
        out = self.zeros() if out is None else out
        sites = np.ascontiguousarray(sites, dtype=np.int64)
        self.lib.orc_s_affine(self.V4, self.L5, self.mf, a, b, _p(v), _p(out), _p(sites), len(sites), int(dagger))
        return out

    def Lam(self, v, sites, dagger=False):
        return self.s_affine(0.0, 1.0, v, sites, dagger)

    def A(self, v, sites, dagger=False):
        return self.s_affine(self.alpha, self.beta, v, sites, dagger)

    def B(self, v, sites, dagger=False):
        return self.s_affine(self.b5, self.c5, v, sites, dagger)

    def Ainv(self, v, sites, dagger=False, out=None):
        out = self.zeros() if out is None else out
        sites = np.ascontiguousarray(sites, dtype=np.int64)
        self.lib.orc_Ainv(self.V4, self.L5, self.alpha, self.beta, self.mf, _p(v), _p(out), _p(sites),
                          len(sites), int(dagger))
        return out

    def axpby(self, a, x, b, y, sites):
        out = self.zeros()
        sites = np.ascontiguousarray(sites, dtype=np.int64)
        self.lib.orc_axpby(self.V4, self.L5, a, _p(x), b, _p(y), _p(out), _p(sites), len(sites))
        return out

    def redot(self, x, y, sites):
        sites = np.ascontiguousarray(sites, dtype=np.int64)
        return float(self.lib.orc_redot(self.V4, self.L5, _p(x), _p(y), _p(sites), len(sites)))

    # ---- D4 / D6: Wilson kernel and the 5D Moebius operator on the full lattice ------
    def DW(self, v):
        """D4: D_W = (4 - M5) - H/2, applied to every s-slice."""
        return (4.0 - self.M5) * v - 0.5 * self.hop(v, self.sites_all)

    def D(self, v):
        """D6: D v = A v - (1/2) H (B v)."""
        Bv = self.B(v, self.sites_all)
        HBv = self.hop(Bv, self.sites_all)
        Av = self.A(v, self.sites_all)
        return Av - 0.5 * HBv

    def Ddag(self, v):
        """D^+ v = A^+ v - (1/2) B^+ (H^+ v)."""
        Hv = self.hop(v, self.sites_all, dagger=True)
        BHv = self.B(Hv, self.sites_all, dagger=True)
        Av = self.A(v, self.sites_all, dagger=True)
        return Av - 0.5 * BHv

    # ---- D7: even-odd blocks and the asymmetric Schur complement ---------------------
    def D_eo(self, v_o):
        """D_eo v_o = -(1/2) H_eo B v_o (result on even sites)."""
        Bv = self.B(v_o, self.sites_odd)
        return -0.5 * self.hop(Bv, self.sites_even)

    def D_oe(self, v_e):
        Bv = self.B(v_e, self.sites_even)
        return -0.5 * self.hop(Bv, self.sites_odd)

    def Mpc(self, v_o, sites_o=None):
        """Mpc v_o = A v_o - (1/4) H_oe B A^{-1} H_eo B v_o, evaluated on sites_o (default: all odd sites)."""
        if sites_o is None:
            sites_o, sites_e, sites_o2 = self.sites_odd, self.sites_even, self.sites_odd
        else:
            sites_o = np.ascontiguousarray(sites_o, dtype=np.int64)
            sites_e = self.neighbours(sites_o)      # even sites feeding the outputs
            sites_o2 = self.neighbours(sites_e)     # odd sites feeding those
        t1 = self.B(v_o, sites_o2)                  # B v_o
        t2 = self.hop(t1, sites_e)                  # H_eo B v_o
        t3 = self.Ainv(t2, sites_e)                 # A^{-1} H_eo B v_o
        t4 = self.B(t3, sites_e)                    # B A^{-1} H_eo B v_o
        t5 = self.hop(t4, sites_o)                  # H_oe B A^{-1} H_eo B v_o
        t6 = self.A(v_o, sites_o)                   # A v_o
        return self.axpby(1.0, t6, -0.25, t5, sites_o)

    def Mpcdag(self, v_o, sites_o=None):
        """Mpc^+ v_o = A^+ v_o - (1/4) B^+ H'_oe A^{-+} B^+ H'_eo v_o, H' = H^+ = gamma5 H gamma5."""
        if sites_o is None:
            sites_o, sites_e = self.sites_odd, self.sites_even
        else:
            sites_o = np.ascontiguousarray(sites_o, dtype=np.int64)
            sites_e = self.neighbours(sites_o)
        t1 = self.hop(v_o, sites_e, dagger=True)    # H'_eo v_o
        t2 = self.B(t1, sites_e, dagger=True)       # B^+ ...
        t3 = self.Ainv(t2, sites_e, dagger=True)    # A^{-+} ...
        t4 = self.hop(t3, sites_o, dagger=True)     # H'_oe ...
        t5 = self.B(t4, sites_o, dagger=True)       # B^+ ...
        t6 = self.A(v_o, sites_o, dagger=True)      # A^+ v_o
        return self.axpby(1.0, t6, -0.25, t5, sites_o)

    def Mpc_at_sites(self, v_o, sites_o, dagger=False):
        """Mpc (or Mpc^+) evaluated only on the listed odd 4D sites (all s); returns [s][n][4][3]."""
        sites_o = np.ascontiguousarray(sites_o, dtype=np.int64)
        full = self.Mpcdag(v_o, sites_o) if dagger else self.Mpc(v_o, sites_o)
        return np.ascontiguousarray(full.reshape(self.L5, self.V4, 4, 3)[:, sites_o])

    # ---- D8: Schur preparation / reconstruction --------------------------------------
    def parity_part(self, v, parity):
        out = self.zeros()
        s = self.sites(parity)
        out.reshape(self.L5, self.V4, 12)[:, s] = v.reshape(self.L5, self.V4, 12)[:, s]
        return out

    def schur_prepare(self, b):
        """b'_o = b_o - D_oe A^{-1} b_e."""
        b_e = self.parity_part(b, 0)
        b_o = self.parity_part(b, 1)
        return b_o - self.D_oe(self.Ainv(b_e, self.sites_even))

    def schur_reconstruct(self, b, x_o):
        """x_e = A^{-1} (b_e - D_eo x_o); returns the full-lattice x = x_e + x_o."""
        b_e = self.parity_part(b, 0)
        x_e = self.Ainv(b_e - self.D_eo(x_o), self.sites_even)
        return x_e + x_o

    # ---- D9: CG on the normal equations, CGLS recurrences ----------------------------
    def cgls(self, bprime, tol, maxiter, callback=None):
        """Solve Mpc x = b' in the least-squares sense.  Returns x, iterations, residual history ||rho_k||/||b'||."""
        so = self.sites_odd
        x = self.zeros()
        rho = bprime.copy()
        g = self.Mpcdag(rho)
        p = g.copy()
        gam = self.redot(g, g, so)
        bnorm = np.sqrt(self.redot(bprime, bprime, so))
        hist = [1.0]
        k = 0
        if bnorm == 0.0:
            return x, 0, hist
        while k < maxiter:
            q = self.Mpc(p)
            a = gam / self.redot(q, q, so)
            x += a * p
            rho -= a * q
            k += 1
            rn = np.sqrt(self.redot(rho, rho, so)) / bnorm
            hist.append(rn)
            if callback is not None:
                callback(k, x, rho)
            if rn <= tol:
                break
            g = self.Mpcdag(rho)
            gam_new = self.redot(g, g, so)
            p = g + (gam_new / gam) * p
            gam = gam_new
        return x, k, hist

    def solve(self, b, tol=1e-10, maxiter=10000):
        """D8 + D9: x = D^{-1} b through the even-odd Schur system; returns x, iterations, ||b - D x||/||b||."""
        bp = self.schur_prepare(b)
        bnorm = np.sqrt(self.redot(b, b, self.sites_all))
        bpn = np.sqrt(self.redot(bp, bp, self.sites_odd))
        inner_tol = tol if bpn == 0 else min(tol, tol * bnorm / bpn)
        x_o, iters, _ = self.cgls(bp, inner_tol, maxiter)
        x = self.schur_reconstruct(b, x_o)
        return x, iters, self.true_residual(b, x)

    def true_residual(self, b, x):
        r = b - self.D(x)
        return float(np.sqrt(self.redot(r, r, self.sites_all) / self.redot(b, b, self.sites_all)))

    # =====================================================================================================
    # 4D <-> 5D maps (Eq. (5), defines the physical quark field q(x)
    # on the walls and the midpoint field of the residual-mass ratio).  4D fields are eta[t][z][y][x][4][3].
    # Readings (N1-N3): chirality convention of D5 (P- lives on s = 0, P+ on s = L5-1 for q);
    # the source is injected on the opposite chiralities and lifted with D_- = c5 D_W - 1.
    # =====================================================================================================
    def _P(self, v, sign):
        """P+ (sign = +1) or P- (sign = -1) = (1 +- gamma5)/2 with gamma5 = diag(+,+,-,-): keeps spins 0,1 or 2,3."""
        out = np.zeros_like(v)
        if sign > 0:
            out[..., 0:2, :] = v[..., 0:2, :]
        else:
            out[..., 2:4, :] = v[..., 2:4, :]
        return out

    def wall_source(self, eta):
        """b(x,s) = delta_{s,0} P+ eta(x) + delta_{s,L5-1} P- eta(x)."""
        b = self.zeros()
        b[0] += self._P(eta, +1)
        b[self.L5 - 1] += self._P(eta, -1)
        return b

    def Dminus(self, v):
        """D_- v = (c5 D_W - 1) v, slice by slice (D6)."""
        return self.c5 * self.DW(v) - v

    def lift(self, eta):
        """5D source of the physical 4D propagator: D_- applied to the wall source."""
        return self.Dminus(self.wall_source(eta))

    def wall_project(self, psi):
        """q(x) = P- psi(x,0) + P+ psi(x,L5-1)   (the quark field of Eq. (5))."""
        return self._P(psi[0], -1) + self._P(psi[self.L5 - 1], +1)

    def midpoint(self, psi):
        """Q(x) = P- psi(x,L5/2) + P+ psi(x,L5/2-1): the wall fields moved to the middle of the fifth dimension."""
        h = self.L5 // 2
        return self._P(psi[h], -1) + self._P(psi[h - 1], +1)

    # =====================================================================================================
    # symmetric even-odd preconditioning.
    #   Mpc_sym = 1 - (1/4) A^{-1} H_oe B A^{-1} H_eo B          (D7, last line)
    #   Mpc_sym^+ = 1 - (1/4) B^+ H'_oe A^{-+} B^+ H'_eo A^{-+}
    # Schur system: Mpc_sym x_o = A^{-1} b'_o with the same b' and the same reconstruction as D8.
    # =====================================================================================================
    def Mpc_sym(self, v_o):
        so, se = self.sites_odd, self.sites_even
        t1 = self.B(v_o, so)                        # B v_o
        t2 = self.hop(t1, se)                       # H_eo B v_o
        t3 = self.Ainv(t2, se)                      # A^{-1} H_eo B v_o
        t4 = self.B(t3, se)                         # B A^{-1} H_eo B v_o
        t5 = self.hop(t4, so)                       # H_oe B A^{-1} H_eo B v_o
        t6 = self.Ainv(t5, so)                      # A^{-1} H_oe B A^{-1} H_eo B v_o
        return self.axpby(1.0, v_o, -0.25, t6, so)

    def Mpc_sym_dag(self, v_o):
        so, se = self.sites_odd, self.sites_even
        t0 = self.Ainv(v_o, so, dagger=True)        # A^{-+} v_o
        t1 = self.hop(t0, se, dagger=True)          # H'_eo ...
        t2 = self.B(t1, se, dagger=True)            # B^+ ...
        t3 = self.Ainv(t2, se, dagger=True)         # A^{-+} ...
        t4 = self.hop(t3, so, dagger=True)          # H'_oe ...
        t5 = self.B(t4, so, dagger=True)            # B^+ ...
        return self.axpby(1.0, v_o, -0.25, t5, so)

    def cgls_op(self, M, Mdag, rhs, tol_abs, maxiter):
        """D9 for a general operator pair on odd sites; stops on ||rho|| <= tol_abs.  Returns x, iterations."""
        so = self.sites_odd
        x = self.zeros()
        rho = rhs.copy()
        g = Mdag(rho)
        p = g.copy()
        gam = self.redot(g, g, so)
        k = 0
        while k < maxiter and np.sqrt(self.redot(rho, rho, so)) > tol_abs:
            q = M(p)
            a = gam / self.redot(q, q, so)
            x += a * p
            rho -= a * q
            k += 1
            g = Mdag(rho)
            gam_new = self.redot(g, g, so)
            p = g + (gam_new / gam) * p
            gam = gam_new
        return x, k

    def solve_sym(self, b, tol=1e-10, maxiter=10000):
        """x = D^{-1} b through the symmetric Schur system; returns x, iterations, ||b - D x||/||b||."""
        bp = self.schur_prepare(b)
        rhs = self.Ainv(bp, self.sites_odd)
        bnorm = np.sqrt(self.redot(b, b, self.sites_all))
        # ||b' - Mpc x|| = ||A rho|| <= (|alpha| + |beta|) ||rho||: stop on the bound
        x_o, iters = self.cgls_op(self.Mpc_sym, self.Mpc_sym_dag, rhs, tol * bnorm / (abs(self.alpha) + abs(self.beta)), maxiter)
        x = self.schur_reconstruct(b, x_o)
        return x, iters, self.true_residual(b, x)
