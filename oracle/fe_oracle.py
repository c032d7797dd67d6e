"""Python face of the CPU oracle (TEST INFRASTRUCTURE ONLY -- see oracle/fe_oracle.c).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this module.  It never imports the CUDA package and shares no code with it.

The heavy loops (Landau polynomial, gradient stencil and energy, __float128 tensor, O(N^2) field
sum) live in fe_oracle.c; this file composes them in the paper's order:

    rhs   = L * active * (E_Land + E_Grad + E_elec + E_Ext)        PAPER.md:33 (Eq. 1), reading O5
    step  = Euler / Heun / classical RK4 with fixed dt            PAPER.md:117-119, reading O6
    energy= F_Land + F_Grad + F_Elec + F_Ext                      PAPER.md:37 (Eq. 2), 66 (Eq. 5), 80 (Eq. 7)

`field_fft` is the oracle-FFT variant O8: the same K table, plain zero-padded numpy.fft
convolution (a library FFT as one step), no pruning, no symmetry tricks.  It is pinned to the
direct sum in tests/test_oracle_electrostatics.py and used where O(N^2) is too slow.
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess
from dataclasses import dataclass, field
from typing import List, Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fe_oracle.c")
_LIB = os.path.join(_HERE, "libfe_oracle.so")

TERM_LANDAU, TERM_GRADIENT, TERM_ELEC, TERM_EXT, TERM_ALL = 1, 2, 4, 8, 15
EULER, HEUN, RK4 = 0, 1, 2


def build(force: bool = False) -> str:
    """Compile fe_oracle.c with gcc (no fast-math; OpenMP on the independent-output loops)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC,
               "-lquadmath", "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _CLandau(ctypes.Structure):
    _fields_ = [("a1", ctypes.c_double * 3)] + [(k, ctypes.c_double) for k in
                ("a11", "a12", "a111", "a112", "a123", "a1111", "a1112", "a1122", "a1123")] + \
               [("active", ctypes.c_int32)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.orc_landau_f.restype = ctypes.c_double
        _lib.orc_landau_energy_sum.restype = ctypes.c_double
        _lib.orc_grad_energy_sum.restype = ctypes.c_double
        _lib.orc_newell_entry.restype = ctypes.c_double
        _lib.orc_tensor_table.restype = ctypes.c_int
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _ip(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int))


def _c_landau(m) -> _CLandau:
    c = _CLandau()
    c.a1[0], c.a1[1], c.a1[2] = m.a1
    for k in ("a11", "a12", "a111", "a112", "a123", "a1111", "a1112", "a1122", "a1123"):
        setattr(c, k, float(getattr(m, k)))
    c.active = int(m.active)
    return c


@dataclass
class Problem:
    """One simulation.  materials: objects with the fields of fe_inputs.Landau; g: fields of
    fe_inputs.Globals.  Arrays are float64 [3][nz][ny][nx]."""
    n: Tuple[int, int, int]
    d: Tuple[float, float, float]
    periodic: Tuple[int, int, int]
    pbc_images: Tuple[int, int, int]
    materials: Sequence
    g: object
    matmap: Optional[np.ndarray] = None
    zero_mode: bool = True

    def __post_init__(self):
        nx, ny, nz = self.n
        if self.matmap is None:
            self.matmap = np.zeros((nz, ny, nx), dtype=np.uint8)
        self.matmap = np.ascontiguousarray(self.matmap, dtype=np.uint8)
        self._cm = (_CLandau * len(self.materials))(*[_c_landau(m) for m in self.materials])
        self.active = np.ascontiguousarray(
            np.array([int(m.active) for m in self.materials], dtype=np.uint8)[self.matmap])

    @property
    def N(self) -> int:
        return self.n[0] * self.n[1] * self.n[2]

    @property
    def V(self) -> float:
        return self.d[0] * self.d[1] * self.d[2]

    @property
    def shape(self):
        return (3, self.n[2], self.n[1], self.n[0])


def _args(p: Problem):
    n = np.array(p.n, dtype=np.int32)
    d = np.array(p.d, dtype=np.float64)
    per = np.array(p.periodic, dtype=np.int32)
    return n, d, per


# ---------------------------------------------------------------- O1 Landau
def landau_f(m, P3: Sequence[float]) -> float:
    c = _c_landau(m)
    v = np.array(P3, dtype=np.float64)
    return lib().orc_landau_f(ctypes.byref(c), _dp(v))


def landau_dfdp(m, P3: Sequence[float]) -> np.ndarray:
    c = _c_landau(m)
    v = np.array(P3, dtype=np.float64)
    out = np.zeros(3)
    lib().orc_landau_dfdp(ctypes.byref(c), _dp(v), _dp(out))
    return out


def landau_field(p: Problem, P: np.ndarray) -> np.ndarray:
    P = np.ascontiguousarray(P, dtype=np.float64)
    E = np.empty_like(P)
    lib().orc_landau_field(p._cm, p.matmap.ctypes.data_as(ctypes.c_void_p), ctypes.c_int64(p.N), _dp(P), _dp(E))
    return E


def landau_energy(p: Problem, P: np.ndarray) -> float:
    P = np.ascontiguousarray(P, dtype=np.float64)
    return p.V * lib().orc_landau_energy_sum(p._cm, p.matmap.ctypes.data_as(ctypes.c_void_p),
                                             ctypes.c_int64(p.N), _dp(P))


# ---------------------------------------------------------------- O2 gradient
def grad_field(p: Problem, P: np.ndarray) -> np.ndarray:
    P = np.ascontiguousarray(P, dtype=np.float64)
    n, d, per = _args(p)
    E = np.empty_like(P)
    g = p.g
    lib().orc_grad_field(_ip(n), _dp(d), _ip(per), p.active.ctypes.data_as(ctypes.c_void_p), _dp(P),
                         ctypes.c_double(g.G11), ctypes.c_double(g.G12), ctypes.c_double(g.G44),
                         ctypes.c_double(g.G44p), _dp(E))
    return E


def grad_energy(p: Problem, P: np.ndarray) -> float:
    P = np.ascontiguousarray(P, dtype=np.float64)
    n, d, per = _args(p)
    g = p.g
    return p.V * lib().orc_grad_energy_sum(_ip(n), _dp(d), _ip(per), p.active.ctypes.data_as(ctypes.c_void_p),
                                           _dp(P), ctypes.c_double(g.G11), ctypes.c_double(g.G12),
                                           ctypes.c_double(g.G44), ctypes.c_double(g.G44p))


# ---------------------------------------------------------------- O3 tensor and field
COMPS = ("xx", "yy", "zz", "xy", "xz", "yz")


def newell_entry(comp: int, offset: Sequence[int], d: Sequence[float]) -> float:
    """N_comp at integer cell offset (i,j,k): the plain 27-term closed form in __float128."""
    dd = np.array(d, dtype=np.float64)
    return lib().orc_newell_entry(int(comp), int(offset[0]), int(offset[1]), int(offset[2]), _dp(dd))


def table_shape(p: Problem):
    T = [p.n[a] if p.periodic[a] else 2 * p.n[a] - 1 for a in range(3)]
    return (6, T[2], T[1], T[0])


def tensor_table(p: Problem) -> np.ndarray:
    """K[6][Tz][Ty][Tx]: signed offsets on open axes (index d + n - 1), circular index on periodic
    axes (minimum image + image sum + zero-mode rule), see orc_tensor_table."""
    n, d, per = _args(p)
    img = np.array(p.pbc_images, dtype=np.int32)
    K = np.zeros(table_shape(p), dtype=np.float64)
    rc = lib().orc_tensor_table(_ip(n), _dp(d), _ip(per), _ip(img), ctypes.c_int(1 if p.zero_mode else 0), _dp(K))
    if rc != 0:
        raise ValueError("orc_tensor_table: bad arguments")
    return K


def field_direct(p: Problem, K: np.ndarray, P: np.ndarray, targets: Optional[np.ndarray] = None) -> np.ndarray:
    """E_elec by summation over all cell pairs (O3).  targets: linear cell indices -> E[3][len]."""
    P = np.ascontiguousarray(P, dtype=np.float64)
    K = np.ascontiguousarray(K, dtype=np.float64)
    n, d, per = _args(p)
    scale = 1.0 / (p.g.eps0 * p.g.epsB)
    if targets is None:
        E = np.empty_like(P)
        lib().orc_field_direct(_ip(n), _ip(per), _dp(K), _dp(P), ctypes.c_double(scale),
                               ctypes.c_int64(0), None, _dp(E))
        return E
    t = np.ascontiguousarray(targets, dtype=np.int64)
    E = np.empty((3, t.size), dtype=np.float64)
    lib().orc_field_direct(_ip(n), _ip(per), _dp(K), _dp(P), ctypes.c_double(scale),
                           ctypes.c_int64(t.size), t.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)), _dp(E))
    return E


_CIDX = ((0, 3, 4), (3, 1, 5), (4, 5, 2))


def circular_kernel(p: Problem, K: np.ndarray) -> np.ndarray:
    """The K table laid out on the zero-padded box [6][mz][my][mx] (m = 2n open, n periodic):
    entry at index (d mod m) holds K(d); index n of an open axis (never a pair offset) is 0."""
    m = [p.n[a] if p.periodic[a] else 2 * p.n[a] for a in range(3)]
    box = np.zeros((6, m[2], m[1], m[0]))
    idx = []
    for a in range(3):
        if p.periodic[a]:
            idx.append(np.arange(p.n[a]))
        else:
            idx.append(np.arange(-(p.n[a] - 1), p.n[a]) % m[a])
    box[np.ix_(range(6), idx[2], idx[1], idx[0])] = K
    return box


def _fftn(a: np.ndarray, axes, workers: Optional[int]):
    """The library FFT used as one step of O8: numpy.fft, or -- when the caller asks for host threads (bench.py's
    all-cores CPU baseline) -- scipy.fft with that many workers.  Same transform, same padding."""
    if workers is None:
        return np.fft.fftn(a, axes=axes)
    import scipy.fft
    return scipy.fft.fftn(a, axes=axes, workers=workers)


def _ifftn(a: np.ndarray, workers: Optional[int]):
    if workers is None:
        return np.fft.ifftn(a)
    import scipy.fft
    return scipy.fft.ifftn(a, workers=workers)


def field_fft(p: Problem, K: np.ndarray, P: np.ndarray, box_hat: Optional[np.ndarray] = None,
              workers: Optional[int] = None) -> np.ndarray:
    """O8: E_elec = -scale * IFFT( FFT(K_box) * FFT(P zero-padded) ), cropped.  Complex transforms
    of the whole padded box; the result's imaginary part is rounding noise and is dropped."""
    nx, ny, nz = p.n
    m = [p.n[a] if p.periodic[a] else 2 * p.n[a] for a in range(3)]
    if box_hat is None:
        box_hat = _fftn(circular_kernel(p, K), (1, 2, 3), workers)
    Pp = np.zeros((3, m[2], m[1], m[0]))
    Pp[:, :nz, :ny, :nx] = P
    Ph = _fftn(Pp, (1, 2, 3), workers)
    scale = 1.0 / (p.g.eps0 * p.g.epsB)
    E = np.empty((3, nz, ny, nx))
    for i in range(3):
        acc = sum(box_hat[_CIDX[i][j]] * Ph[j] for j in range(3))
        E[i] = -scale * _ifftn(acc, workers).real[:nz, :ny, :nx]
    return E


# ---------------------------------------------------------------- O5-O7
# Cash-Karp tableau (Cash & Karp 1990): a_ij, 5th-order weights, embedded 4th-order weights
RK45_C = (0.0, 1.0 / 5.0, 3.0 / 10.0, 3.0 / 5.0, 1.0, 7.0 / 8.0)
RK45_A = ((),
          (1.0 / 5.0,),
          (3.0 / 40.0, 9.0 / 40.0),
          (3.0 / 10.0, -9.0 / 10.0, 6.0 / 5.0),
          (-11.0 / 54.0, 5.0 / 2.0, -70.0 / 27.0, 35.0 / 27.0),
          (1631.0 / 55296.0, 175.0 / 512.0, 575.0 / 13824.0, 44275.0 / 110592.0, 253.0 / 4096.0))
RK45_B5 = (37.0 / 378.0, 0.0, 250.0 / 621.0, 125.0 / 594.0, 0.0, 512.0 / 1771.0)
RK45_B4 = (2825.0 / 27648.0, 0.0, 18575.0 / 48384.0, 13525.0 / 55296.0, 277.0 / 14336.0, 1.0 / 4.0)


class Oracle:
    """RHS / step / energy of one simulation.  elec = 'direct' (O3) or 'fft' (O8)."""

    def __init__(self, p: Problem, elec: str = "direct", K: Optional[np.ndarray] = None,
                 fft_workers: Optional[int] = None):
        self.p = p
        self.elec = elec
        self.K = K
        self.fft_workers = fft_workers      # None: numpy.fft (single thread); n: scipy.fft with n host threads
        self._box_hat = None
        self.wave = None        # (amp[3], omega, phase): E_ext(t) = g.E_ext + amp sin(omega t + phase)

    def set_wave(self, amp, omega: float, phase: float = 0.0):
        """Time-dependent external excitation: a sinusoid added to the static field."""
        self.wave = (np.array(amp, dtype=np.float64), float(omega), float(phase))

    def e_ext(self, t: float = 0.0) -> np.ndarray:
        E = np.array(self.p.g.E_ext, dtype=np.float64)
        if self.wave is not None:
            amp, om, ph = self.wave
            E = E + amp * math.sin(om * t + ph)
        return E

    def table(self) -> np.ndarray:
        if self.K is None:
            self.K = tensor_table(self.p)
        return self.K

    def elec_field(self, P: np.ndarray) -> np.ndarray:
        K = self.table()
        if self.elec == "direct":
            return field_direct(self.p, K, P)
        if self._box_hat is None:
            self._box_hat = _fftn(circular_kernel(self.p, K), (1, 2, 3), self.fft_workers)
        return field_fft(self.p, K, P, self._box_hat, self.fft_workers)

    def fields(self, P: np.ndarray, terms: int = TERM_ALL, t: float = 0.0):
        p = self.p
        z = np.zeros(p.shape)
        El = landau_field(p, P) if terms & TERM_LANDAU else z
        Eg = grad_field(p, P) if terms & TERM_GRADIENT else z
        Ee = self.elec_field(P) if terms & TERM_ELEC else z
        Ex = (self.e_ext(t)[:, None, None, None] * np.ones(p.shape)
              if terms & TERM_EXT else z)
        return El, Eg, Ee, Ex

    def rhs(self, P: np.ndarray, terms: int = TERM_ALL, t: float = 0.0) -> np.ndarray:
        El, Eg, Ee, Ex = self.fields(P, terms, t)
        return self.p.g.L * self.p.active[None] * (El + Eg + Ee + Ex)

    def step(self, P: np.ndarray, dt: float, nsteps: int = 1, integrator: int = EULER,
             terms: int = TERM_ALL, t0: float = 0.0) -> np.ndarray:
        """Step n goes from t0 + n dt to t0 + (n + 1) dt; the stages sample E_ext at the usual abscissae."""
        P = np.array(P, dtype=np.float64, copy=True)
        f = lambda Y, t: self.rhs(Y, terms, t)
        for n in range(nsteps):
            t = t0 + n * dt
            if integrator == EULER:
                P = P + dt * f(P, t)
            elif integrator == HEUN:
                k1 = f(P, t)
                k2 = f(P + dt * k1, t + dt)
                P = P + (dt / 2.0) * (k1 + k2)
            elif integrator == RK4:
                k1 = f(P, t)
                k2 = f(P + (dt / 2.0) * k1, t + dt / 2.0)
                k3 = f(P + (dt / 2.0) * k2, t + dt / 2.0)
                k4 = f(P + dt * k3, t + dt)
                P = P + dt * (k1 / 6.0 + k2 / 3.0 + k3 / 3.0 + k4 / 6.0)
            else:
                raise ValueError("integrator")
        return P

    def step_ab3m2(self, P: np.ndarray, dt: float, nsteps: int, terms: int = TERM_ALL, t0: float = 0.0) -> np.ndarray:
        """AB3M2 ("Adams-Bashforth (AB3M2), a multistep explicit scheme", ref. [53]), reading A18:
        predictor = 3-step Adams-Bashforth, corrector = 2nd-order Adams-Moulton (trapezoid), one correction (PECE);
        the first two steps, which have no history, are Heun steps:
            P*      = P_n + dt/12 (23 f_n - 16 f_{n-1} + 5 f_{n-2})
            P_{n+1} = P_n + dt/2  (f_n + f(P*))"""
        P = np.array(P, dtype=np.float64, copy=True)
        f = lambda Y, t: self.rhs(Y, terms, t)
        hist = []                                    # f_{n-1}, f_{n-2}
        for n in range(nsteps):
            t = t0 + n * dt
            fn = f(P, t)
            if n < 2:
                Pstar = P + dt * fn
            else:
                Pstar = P + (dt / 12.0) * (23.0 * fn - 16.0 * hist[0] + 5.0 * hist[1])
            P = P + (dt / 2.0) * (fn + f(Pstar, t + dt))
            hist = [fn] + hist[:1]
        return P

    def step_rk45(self, P: np.ndarray, t_span: float, dt_init: float, tol: float, max_steps: int = 100000,
                  terms: int = TERM_ALL, t0: float = 0.0):
        """Adaptive RK45 (ref. [52] "fifth order Runge-Kutta with adaptive step size control"), reading
        A17: the Cash-Karp embedded pair; the 5th-order solution is propagated, err = max over cells and components
        of |y5 - y4| / tol (absolute tolerance, state units); a step is accepted when err <= 1,
            accepted: dt_next = 0.9 dt err^-0.2  (5 dt when err <= 1.89e-4),
            rejected: dt      = max(0.9 dt err^-0.25, 0.1 dt);
        the last step is shortened to land on t_span.  Returns (P, stats)."""
        P = np.array(P, dtype=np.float64, copy=True)
        f = lambda Y, tt: self.rhs(Y, terms, tt)
        A, B5, B4, C = RK45_A, RK45_B5, RK45_B4, RK45_C
        t, dt = 0.0, float(dt_init)
        acc = rej = evals = 0
        err = 0.0
        dt_last = 0.0
        while t < t_span and acc + rej < max_steps:
            h = min(dt, t_span - t)
            k = []
            for i in range(6):
                Y = P.copy()
                for j in range(i):
                    if A[i][j] != 0.0:
                        Y = Y + (h * A[i][j]) * k[j]
                k.append(f(Y, t0 + t + C[i] * h))
            evals += 6
            y5 = P.copy()
            d = np.zeros_like(P)
            for j in range(6):
                if B5[j] != 0.0:
                    y5 = y5 + (h * B5[j]) * k[j]
                d = d + (h * (B5[j] - B4[j])) * k[j]
            err = float(np.max(np.abs(d))) / tol
            if err <= 1.0:
                P, t, acc, dt_last = y5, t + h, acc + 1, h
                dt = 5.0 * h if err <= 1.89e-4 else 0.9 * h * err ** -0.2
            else:
                rej += 1
                dt = max(0.9 * h * err ** -0.25, 0.1 * h)
        return P, dict(t=t, accepted=acc, rejected=rej, rhs_evals=evals, dt_last=dt_last, dt_next=dt, err_last=err)

    def energy(self, P: np.ndarray, terms: int = TERM_ALL) -> np.ndarray:
        """[F_Land, F_Grad, F_Elec, F_Ext, F_tot, <Px>, <Py>, <Pz>] (means over active cells)."""
        p = self.p
        FL = landau_energy(p, P) if terms & TERM_LANDAU else 0.0
        FG = grad_energy(p, P) if terms & TERM_GRADIENT else 0.0
        FE = -0.5 * p.V * float(np.sum(self.elec_field(P) * P)) if terms & TERM_ELEC else 0.0
        FX = (-p.V * float(sum(p.g.E_ext[i] * np.sum(P[i]) for i in range(3)))
              if terms & TERM_EXT else 0.0)
        na = max(int(p.active.sum()), 1)
        mean = [float(np.sum(P[i] * p.active)) / na for i in range(3)]
        return np.array([FL, FG, FE, FX, FL + FG + FE + FX, *mean])
