"""CPU oracle for the neural DSMC collision step -- TEST INFRASTRUCTURE, not product.

Thin ctypes marshalling around ``oracle/dsmc_oracle.c`` (plain C99, fp64, single thread,
written from /root/reference/PAPER.md; see that file and DESIGN.md for citations and
readings).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package.  It imports nothing
from ``paper_2602_21244_b200`` and shares no code with the CUDA path.

Parity status: see the header of ``dsmc_oracle.h`` (trained-model behaviour is
"parity unpinned"; everything else is pinned by tests/test_oracle_*.py).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_DIR, "dsmc_oracle.c")
_HDR = os.path.join(_DIR, "dsmc_oracle.h")
_LIB = os.path.join(_DIR, "liboracle.so")

KB = 1.380649e-23

F_NOISE, F_ENERGY_SHELL, F_MOMENT_MATCH, F_ACCEPT, F_MATCH_ENERGY_ONLY = 1, 2, 4, 8, 32
F_PAIR_REPLACE = 128
ACT_TANH, ACT_RELU, ACT_SILU = 0, 1, 2
POT_LJ, POT_HARD_SPHERE, POT_INV_R, POT_INV_R2 = 0, 1, 2, 3


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 (no fast-math).  Building the checker is not using it.
    ORACLE_SANITIZE=1 builds (and loads) an AddressSanitizer + UBSan copy instead; run the tests with
    LD_PRELOAD=$(gcc -print-file-name=libasan.so) (profiles/r02_oracle_asan_ubsan.md)."""
    san = os.environ.get("ORACLE_SANITIZE") == "1"
    lib_path = _LIB.replace(".so", "_san.so") if san else _LIB
    stale = (not os.path.exists(lib_path)) or os.path.getmtime(lib_path) < max(
        os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    if force or stale:
        tmp = lib_path + ".tmp.%d" % os.getpid()
        flags = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
                 "-fno-omit-frame-pointer"] if san else ["-O2"]
        subprocess.check_call(["gcc", *flags, "-std=c99", "-fPIC", "-shared", "-Wall", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, lib_path)
    return lib_path


class _Mlp(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("dims", C.c_int32 * 8), ("act", C.c_int32),
                ("W", C.POINTER(C.c_float) * 7), ("b", C.POINTER(C.c_float) * 7)]


class _Vhs(C.Structure):
    _fields_ = [("mass", C.c_double), ("sigma_v", C.c_double), ("T_scale", C.c_double),
                ("noise_sigma", C.c_double), ("shell_eps", C.c_double), ("d_ref", C.c_double),
                ("omega", C.c_double), ("T_ref", C.c_double), ("pairs_per_cell", C.c_int32),
                ("flags", C.c_uint32), ("cell_base", C.c_int32), ("pairs_count", C.POINTER(C.c_int32))]


class _Abi(C.Structure):
    _fields_ = [("mass", C.c_double), ("b_max", C.c_double), ("lnE_min", C.c_double),
                ("lnE_max", C.c_double), ("chi_mode", C.c_int32), ("pairs_per_cell", C.c_int32),
                ("flags", C.c_uint32), ("cell_base", C.c_int32), ("pairs_count", C.POINTER(C.c_int32))]


class _Table(C.Structure):
    _fields_ = [("chi", C.POINTER(C.c_float)), ("nE", C.c_int32), ("nB", C.c_int32),
                ("lnE_min", C.c_double), ("lnE_max", C.c_double)]


class _Pot(C.Structure):
    _fields_ = [("kind", C.c_int32), ("p0", C.c_double), ("p1", C.c_double), ("r_hi", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_u01.restype = C.c_double
        _lib.orc_pair_key.restype = C.c_uint32
        _lib.orc_pair_key.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32]
        _lib.orc_pairing.restype = C.c_int32
        _lib.orc_vhs_sigma_g.restype = C.c_double
        _lib.orc_chi_bilinear.restype = C.c_double
        _lib.orc_chi_mlp.restype = C.c_double
        _lib.orc_potential_eval.restype = C.c_double
        _lib.orc_rmin.restype = C.c_double
        _lib.orc_chi_exact.restype = C.c_double
    return _lib


def _p(a, ty):
    return a.ctypes.data_as(C.POINTER(ty)) if a is not None else None


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


# ------------------------------------------------------------------------------- parameter objects
@dataclass
class Mlp:
    """weights[l]: float32 [out, in]; biases[l]: float32 [out]."""
    weights: list
    biases: list
    act: int = ACT_TANH

    def c(self):
        self._keep = [np.ascontiguousarray(w, dtype=np.float32) for w in self.weights] + \
                     [np.ascontiguousarray(b, dtype=np.float32) for b in self.biases]
        m = _Mlp()
        L = len(self.weights)
        m.n_layers = L
        m.act = self.act
        m.dims[0] = self.weights[0].shape[1]
        for l in range(L):
            m.dims[l + 1] = self.weights[l].shape[0]
            m.W[l] = _p(self._keep[l], C.c_float)
            m.b[l] = _p(self._keep[L + l], C.c_float)
        return m


@dataclass
class VhsParams:
    mass: float = 6.63e-26
    sigma_v: float = 337.2
    T_scale: float = 273.0
    noise_sigma: float = 0.1
    shell_eps: float = 1e-20
    d_ref: float = 4.17e-10
    omega: float = 0.81
    T_ref: float = 273.0
    pairs_per_cell: int = -1
    flags: int = F_NOISE | F_ENERGY_SHELL | F_MOMENT_MATCH
    cell_base: int = 0
    pairs_count: np.ndarray = None  # per-cell request (int32), overrides pairs_per_cell

    def c(self):
        pc = None
        if self.pairs_count is not None:
            self.pairs_count = _i32(self.pairs_count)
            pc = _p(self.pairs_count, C.c_int32)
        return _Vhs(self.mass, self.sigma_v, self.T_scale, self.noise_sigma, self.shell_eps,
                    self.d_ref, self.omega, self.T_ref, self.pairs_per_cell, self.flags, self.cell_base, pc)


@dataclass
class AbinitioParams:
    mass: float = 6.63e-26
    b_max: float = 1e-9
    lnE_min: float = float(np.log(5.0))
    lnE_max: float = float(np.log(6.0e4))
    chi_mode: int = 0
    pairs_per_cell: int = -1
    flags: int = F_MOMENT_MATCH
    cell_base: int = 0
    pairs_count: np.ndarray = None  # per-cell request (int32), overrides pairs_per_cell

    def c(self):
        pc = None
        if self.pairs_count is not None:
            self.pairs_count = _i32(self.pairs_count)
            pc = _p(self.pairs_count, C.c_int32)
        return _Abi(self.mass, self.b_max, self.lnE_min, self.lnE_max, self.chi_mode,
                    self.pairs_per_cell, self.flags, self.cell_base, pc)


@dataclass
class ChiTable:
    chi: np.ndarray  # float32 [nE, nB]
    lnE_min: float
    lnE_max: float

    def c(self):
        self._keep = np.ascontiguousarray(self.chi, dtype=np.float32)
        return _Table(_p(self._keep, C.c_float), self._keep.shape[0], self._keep.shape[1],
                      self.lnE_min, self.lnE_max)


@dataclass
class Potential:
    kind: int
    p0: float
    p1: float = 0.0
    r_hi: float = 0.0

    def c(self):
        return _Pot(self.kind, self.p0, self.p1, self.r_hi)


def lj_argon() -> Potential:
    """LJ 12-6, eps/k = 119.8 K, sigma = 3.405 A (BASELINE.json cfg 4 fallback, Q17)."""
    return Potential(POT_LJ, 119.8 * KB, 3.405e-10, 10 * 3.405e-10)


# --------------------------------------------------------------------------------------- functions
def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def u01(x):
    return lib().orc_u01(C.c_uint32(int(x)))


def pair_key(seed, step, cell, slot):
    return int(lib().orc_pair_key(int(seed), int(step), int(cell), int(slot)))


def pair_uniforms(seed, step, cell, s):
    u = (C.c_double * 3)()
    lib().orc_pair_uniforms(C.c_uint64(seed), C.c_uint32(step), C.c_uint32(cell), C.c_uint32(s), u)
    return np.array(list(u))


def pair_uniforms_batch(seed, step, cells, slots):
    """(U_acc, U_b, U_eps) of many (cell, pair slot): array [n, 3]."""
    cells = np.ascontiguousarray(cells, np.uint32)
    slots = np.ascontiguousarray(slots, np.uint32)
    u = np.empty((cells.shape[0], 3), np.float64)
    lib().orc_pair_uniforms_batch(C.c_uint64(seed), C.c_uint32(step), C.c_int64(cells.shape[0]),
                                  _p(cells, C.c_uint32), _p(slots, C.c_uint32), _p(u, C.c_double))
    return u


def pair_draw(seed, step, cell, s, N):
    i, j = C.c_int32(0), C.c_int32(0)
    lib().orc_pair_draw(C.c_uint64(seed), C.c_uint32(step), C.c_uint32(cell), C.c_uint32(s), C.c_int32(N), C.byref(i), C.byref(j))
    return i.value, j.value


def pair_normals(seed, step, cell, s):
    u = (C.c_double * 3)()
    lib().orc_pair_normals(C.c_uint64(seed), C.c_uint32(step), C.c_uint32(cell), C.c_uint32(s), u)
    return np.array(list(u))


def bin_particles(cell, n_cells):
    cell = _i32(cell)
    n = cell.shape[0]
    perm = np.empty(n, np.int32)
    cell_start = np.empty(n_cells + 1, np.int32)
    rc = lib().orc_bin(C.c_int64(n), C.c_int32(n_cells), _p(cell, C.c_int32), _p(perm, C.c_int32),
                       _p(cell_start, C.c_int32))
    return rc, perm, cell_start


def cell_moments(cell_start, vx, vy, vz):
    cell_start = _i32(cell_start)
    K = cell_start.shape[0] - 1
    vx, vy, vz = _f64(vx), _f64(vy), _f64(vz)
    out = np.empty((K, 4), np.float64)
    lib().orc_cell_moments(C.c_int32(K), _p(cell_start, C.c_int32), _p(vx, C.c_double),
                           _p(vy, C.c_double), _p(vz, C.c_double), _p(out, C.c_double))
    return out


def cell_state(vx, vy, vz, mass):
    vx, vy, vz = _f64(vx), _f64(vy), _f64(vz)
    ubar = (C.c_double * 3)()
    th, T = C.c_double(), C.c_double()
    lib().orc_cell_state(C.c_int64(vx.shape[0]), _p(vx, C.c_double), _p(vy, C.c_double),
                         _p(vz, C.c_double), C.c_double(mass), ubar, C.byref(th), C.byref(T))
    return np.array(list(ubar)), th.value, T.value


def pairing(seed, step, cell, N, M_req=-1):
    pi = np.empty(max(N, 1), np.int32)
    M = lib().orc_pairing(C.c_uint64(seed), C.c_uint32(step), C.c_uint32(cell), C.c_int32(N),
                          C.c_int32(M_req), _p(pi, C.c_int32))
    return int(M), pi[:N]


def pairing_all(seed, step, cell_start, cell_base=0, M_req=-1):
    """The matching of every cell (pairing alone, integer work): (pair_i, pair_j) in the layout of the pair dump."""
    cs = _i32(cell_start)
    n = int(cs[-1])
    pi = np.empty(max(n, 1), np.int32)
    pj = np.empty(max(n, 1), np.int32)
    lib().orc_pairing_all(C.c_uint64(seed), C.c_uint32(step), C.c_int32(cs.shape[0] - 1), _p(cs, C.c_int32),
                          C.c_uint32(cell_base), C.c_int32(M_req), _p(pi, C.c_int32), _p(pj, C.c_int32))
    return pi[:n], pj[:n]


def mlp_forward(net: Mlp, x):
    x = _f64(x)
    out = np.empty(net.weights[-1].shape[0], np.float64)
    m = net.c()
    lib().orc_mlp_forward(C.byref(m), _p(x, C.c_double), _p(out, C.c_double))
    return out


def vhs_sigma_g(g, prm: VhsParams):
    p = prm.c()
    return lib().orc_vhs_sigma_g(C.c_double(g), C.byref(p))


def rotate(g, chi, eps):
    g = _f64(g)
    out = np.empty(3, np.float64)
    lib().orc_rotate(_p(g, C.c_double), C.c_double(chi), C.c_double(eps), _p(out, C.c_double))
    return out


def chi_bilinear(table: ChiTable, lnE, btilde):
    t = table.c()
    return lib().orc_chi_bilinear(C.byref(t), C.c_double(lnE), C.c_double(btilde))


def chi_mlp(net: Mlp, lnE_min, lnE_max, lnE, btilde):
    m = net.c()
    return lib().orc_chi_mlp(C.byref(m), C.c_double(lnE_min), C.c_double(lnE_max), C.c_double(lnE),
                             C.c_double(btilde))


def moment_match(cell_start, vx, vy, vz, target, flags=F_MOMENT_MATCH):
    """Returns new (vx, vy, vz) float64 arrays."""
    cell_start = _i32(cell_start)
    K = cell_start.shape[0] - 1
    vx, vy, vz = _f64(vx).copy(), _f64(vy).copy(), _f64(vz).copy()
    target = _f64(target)
    lib().orc_moment_match(C.c_int32(K), _p(cell_start, C.c_int32), _p(vx, C.c_double),
                           _p(vy, C.c_double), _p(vz, C.c_double), _p(target, C.c_double),
                           C.c_uint32(flags))
    return vx, vy, vz


@dataclass
class StepResult:
    vx: np.ndarray
    vy: np.ndarray
    vz: np.ndarray
    pair_i: np.ndarray
    pair_j: np.ndarray
    accepted: np.ndarray
    gprime: np.ndarray
    aux: np.ndarray  # |h_hat| (VHS-NN) or chi (ab initio), per dump index


def _step_buffers(n):
    return (np.full(n, -1, np.int32), np.full(n, -1, np.int32), np.zeros(n, np.uint8),
            np.zeros((n, 3), np.float64), np.zeros(n, np.float64))


def collide_vhs_nn(cell_start, vx, vy, vz, net: Mlp, prm: VhsParams, seed, step,
                   sigma_cr_max=None) -> StepResult:
    cell_start = _i32(cell_start)
    K = cell_start.shape[0] - 1
    vx, vy, vz = _f64(vx).copy(), _f64(vy).copy(), _f64(vz).copy()
    n = vx.shape[0]
    pi, pj, acc, gp, aux = _step_buffers(n)
    scm = None if sigma_cr_max is None else np.ascontiguousarray(sigma_cr_max, np.float32)
    m, p = net.c(), prm.c()
    rc = lib().orc_collide_vhs_nn(
        C.c_int64(n), C.c_int32(K), _p(cell_start, C.c_int32), _p(vx, C.c_double),
        _p(vy, C.c_double), _p(vz, C.c_double), _p(scm, C.c_float), C.byref(m), C.byref(p),
        C.c_uint64(seed), C.c_uint32(step), _p(pi, C.c_int32), _p(pj, C.c_int32),
        _p(acc, C.c_uint8), _p(gp, C.c_double), _p(aux, C.c_double))
    if rc != 0:
        raise ValueError("orc_collide_vhs_nn rc=%d" % rc)
    return StepResult(vx, vy, vz, pi, pj, acc, gp, aux)


def collide_abinitio(cell_start, vx, vy, vz, prm: AbinitioParams, seed, step, net: Mlp = None,
                     table: ChiTable = None, cr_max=None) -> StepResult:
    cell_start = _i32(cell_start)
    K = cell_start.shape[0] - 1
    vx, vy, vz = _f64(vx).copy(), _f64(vy).copy(), _f64(vz).copy()
    n = vx.shape[0]
    pi, pj, acc, gp, aux = _step_buffers(n)
    crm = None if cr_max is None else np.ascontiguousarray(cr_max, np.float32)
    m = net.c() if net is not None else None
    t = table.c() if table is not None else None
    p = prm.c()
    rc = lib().orc_collide_abinitio(
        C.c_int64(n), C.c_int32(K), _p(cell_start, C.c_int32), _p(vx, C.c_double),
        _p(vy, C.c_double), _p(vz, C.c_double), _p(crm, C.c_float),
        C.byref(m) if m is not None else None, C.byref(t) if t is not None else None, C.byref(p),
        C.c_uint64(seed), C.c_uint32(step), _p(pi, C.c_int32), _p(pj, C.c_int32),
        _p(acc, C.c_uint8), _p(gp, C.c_double), _p(aux, C.c_double))
    if rc != 0:
        raise ValueError("orc_collide_abinitio rc=%d" % rc)
    return StepResult(vx, vy, vz, pi, pj, acc, gp, aux)


def chi_batch(E_over_k, b, chi_mode, b_max, net: Mlp = None, table: ChiTable = None,
              lnE_min=float(np.log(5.0)), lnE_max=float(np.log(6.0e4))):
    E_over_k = np.ascontiguousarray(E_over_k, np.float32)
    b = np.ascontiguousarray(b, np.float32)
    out = np.empty(E_over_k.shape[0], np.float64)
    m = net.c() if net is not None else None
    t = table.c() if table is not None else None
    lib().orc_chi_batch(C.c_int64(out.shape[0]), _p(E_over_k, C.c_float), _p(b, C.c_float),
                        _p(out, C.c_double), C.c_int32(chi_mode),
                        C.byref(m) if m is not None else None,
                        C.byref(t) if t is not None else None, C.c_double(b_max),
                        C.c_double(lnE_min), C.c_double(lnE_max))
    return out


def potential_eval(pot: Potential, r):
    p = pot.c()
    return lib().orc_potential_eval(C.byref(p), C.c_double(r))


def rmin(pot: Potential, E, b):
    p = pot.c()
    return lib().orc_rmin(C.byref(p), C.c_double(E), C.c_double(b))


def chi_exact(pot: Potential, E, b, n_panels=16):
    p = pot.c()
    return lib().orc_chi_exact(C.byref(p), C.c_double(E), C.c_double(b), C.c_int32(n_panels))


def cap_chi(c):
    f = lib().orc_cap_chi
    f.restype = C.c_double
    return float(f(C.c_double(c)))


def build_chi_table(pot: Potential, nE, nB, lnE_min=float(np.log(5.0)),
                    lnE_max=float(np.log(6.0e4)), b_max=1e-9, n_panels=4) -> ChiTable:
    chi = np.empty((nE, nB), np.float32)
    p = pot.c()
    lib().orc_build_chi_table(C.byref(p), C.c_int32(nE), C.c_int32(nB), C.c_double(lnE_min),
                              C.c_double(lnE_max), C.c_double(b_max), C.c_int32(n_panels),
                              _p(chi, C.c_float))
    return ChiTable(chi, lnE_min, lnE_max)


def build_chi_table_mlp(net: Mlp, nE, nB, lnE_min=float(np.log(5.0)), lnE_max=float(np.log(6.0e4))) -> ChiTable:
    """f2: the chi-MLP evaluated on the table nodes."""
    chi = np.empty((nE, nB), np.float32)
    m = net.c()
    lib().orc_build_chi_table_mlp(C.byref(m), C.c_int32(nE), C.c_int32(nB), C.c_double(lnE_min), C.c_double(lnE_max),
                                  _p(chi, C.c_float))
    return ChiTable(chi, lnE_min, lnE_max)


# ------------------------------------------------------------- f4: move + walls + sampling (Q30)
class _Couette(C.Structure):
    _fields_ = [("L", C.c_double), ("dt", C.c_double), ("u_wall", C.c_double), ("rt_wall", C.c_double),
                ("accommodation", C.c_double), ("n_cells", C.c_int32)]


MAX_BOUNCES = 4


@dataclass
class CouetteParams:
    L: float
    dt: float
    u_wall: float
    rt_wall: float
    accommodation: float
    n_cells: int

    def c(self):
        return _Couette(self.L, self.dt, self.u_wall, self.rt_wall, self.accommodation, self.n_cells)


def move_couette(x, vx, vy, vz, prm: CouetteParams, seed, step):
    """Free flight for dt between Maxwell walls (Q30).  Returns (x, vx, vy, vz, cell, bounces, margin)."""
    x, vx, vy, vz = (_f64(a).copy() for a in (x, vx, vy, vz))
    n = x.shape[0]
    cell = np.empty(n, np.int32)
    nb = np.empty(n, np.int32)
    mg = np.empty(n, np.float64)
    c = prm.c()
    lib().orc_move_couette(C.c_int64(n), _p(x, C.c_double), _p(vx, C.c_double), _p(vy, C.c_double),
                           _p(vz, C.c_double), _p(cell, C.c_int32), _p(nb, C.c_int32), _p(mg, C.c_double),
                           C.byref(c), C.c_uint64(seed), C.c_uint32(step))
    return x, vx, vy, vz, cell, nb, mg


def sample_cells(cell_start, vx, vy, vz, acc=None):
    """acc[n_cells, 8] += (count, sums of vx, vy, vz, vx^2, vy^2, vz^2, vx vy) per cell."""
    cs = _i32(cell_start)
    K = cs.shape[0] - 1
    if acc is None:
        acc = np.zeros((K, 8), np.float64)
    vx, vy, vz = _f64(vx), _f64(vy), _f64(vz)
    lib().orc_sample_cells(C.c_int32(K), _p(cs, C.c_int32), _p(vx, C.c_double), _p(vy, C.c_double),
                           _p(vz, C.c_double), _p(acc, C.c_double))
    return acc


def ntc_counts(cell_start, sigma_cr_max, coef, remainder):
    """NTC candidate counts with carried remainder (Q31); `remainder` (float64) is updated in place."""
    cs = _i32(cell_start)
    K = cs.shape[0] - 1
    scm = np.ascontiguousarray(sigma_cr_max, np.float32)
    assert remainder.dtype == np.float64 and remainder.flags.c_contiguous and remainder.shape[0] == K
    counts = np.empty(K, np.int32)
    lib().orc_ntc_counts(C.c_int32(K), _p(cs, C.c_int32), _p(scm, C.c_float), C.c_double(coef),
                         _p(remainder, C.c_double), _p(counts, C.c_int32))
    return counts
