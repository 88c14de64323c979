"""Thin Python binding of libdsmc_b200.so (include/dsmc.h): argument marshalling only.

Same names as the C ABI.  PyTorch is used for device memory and streams; every step of the
path runs in the library's sm_100a kernels.  There is no CPU fallback: importing this module
raises if the shared library is missing, and every call raises ``DsmcError`` on a non-zero status.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np
import torch

_DIR = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_DIR, "libdsmc_b200.so")

OK = 0
ERR_INVALID_ARG, ERR_BAD_CELL_INDEX, ERR_CELL_TOO_LARGE = -1, -2, -3
ERR_NOT_CONFIGURED, ERR_CUDA, ERR_UNSUPPORTED_SHAPE = -4, -5, -6
MAX_CELL_PARTICLES = 2048

F_NOISE, F_ENERGY_SHELL, F_MOMENT_MATCH, F_ACCEPT, F_BF16_TC, F_MATCH_ENERGY_ONLY, F_CHI_ABS = 1, 2, 4, 8, 16, 32, 64
F_PAIR_REPLACE = 128
F_TC_ONE_KERNEL = 256
ACT_TANH, ACT_RELU, ACT_SILU = 0, 1, 2

EXPORTS = ["dsmc_create", "dsmc_destroy", "dsmc_set_stream", "dsmc_sync_status", "dsmc_strerror",
           "dsmc_launch_count", "dsmc_set_mlp", "dsmc_set_chi_table", "dsmc_bin", "dsmc_collide_vhs_nn",
           "dsmc_collide_abinitio", "dsmc_cell_moments", "dsmc_moment_match", "dsmc_chi_batch",
           "dsmc_chi_exact_batch", "dsmc_build_chi_table_lj", "dsmc_build_chi_table_mlp", "dsmc_step_host", "dsmc_step_host_submit", "dsmc_move_couette",
           "dsmc_gather_f32", "dsmc_sample_cells", "dsmc_couette_run", "dsmc_ntc_counts", "dsmc_noalloc_setup", "dsmc_bin_noalloc"]


class DsmcError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        super().__init__("%s failed: %d (%s)" % (where, status, strerror(status)))


class _MlpDesc(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("dims", C.c_int32 * 8), ("act", C.c_int32),
                ("W", C.POINTER(C.POINTER(C.c_float))), ("b", C.POINTER(C.POINTER(C.c_float)))]


class _VhsParams(C.Structure):
    _fields_ = [("mass", C.c_float), ("sigma_v", C.c_float), ("T_scale", C.c_float),
                ("noise_sigma", C.c_float), ("shell_eps", C.c_float), ("d_ref", C.c_float),
                ("omega", C.c_float), ("T_ref", C.c_float), ("pairs_per_cell", C.c_int32),
                ("flags", C.c_uint32), ("cell_base", C.c_int32), ("pairs_count", C.c_void_p)]


class _AbiParams(C.Structure):
    _fields_ = [("mass", C.c_float), ("b_max", C.c_float), ("lnE_min", C.c_float), ("lnE_max", C.c_float),
                ("chi_mode", C.c_int32), ("pairs_per_cell", C.c_int32), ("flags", C.c_uint32),
                ("cell_base", C.c_int32), ("pairs_count", C.c_void_p)]


class _CouetteParams(C.Structure):
    _fields_ = [("L", C.c_float), ("dt", C.c_float), ("u_wall", C.c_float), ("rt_wall", C.c_float),
                ("accommodation", C.c_float), ("n_cells", C.c_int32), ("ntc_coef", C.c_float),
                ("sigma_cr_max", C.c_float)]


class _PairDump(C.Structure):
    _fields_ = [("pair_i", C.c_void_p), ("pair_j", C.c_void_p), ("accepted", C.c_void_p),
                ("gprime", C.c_void_p), ("aux", C.c_void_p)]


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            "libdsmc_b200.so is missing (%s). Build it with `python -m paper_2602_21244_b200.build`; "
            "there is no CPU fallback." % LIB_PATH)
    lib = C.CDLL(LIB_PATH)
    lib.dsmc_strerror.restype = C.c_char_p
    lib.dsmc_launch_count.restype = C.c_int64
    lib.dsmc_launch_count.argtypes = [C.c_void_p]
    return lib


_lib = _load()


def strerror(status: int) -> str:
    return _lib.dsmc_strerror(C.c_int(status)).decode()


def _chk(rc, where):
    if rc != 0:
        raise DsmcError(rc, where)


def _ptr(t, dtype=None):
    if t is None:
        return C.c_void_p(0)
    assert t.is_cuda and t.is_contiguous(), "device, contiguous tensors only"
    if dtype is not None:
        assert t.dtype == dtype, (t.dtype, dtype)
    return C.c_void_p(t.data_ptr())


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
    pairs_count: "torch.Tensor" = None  # device int32 [n_cells]: per-cell request, overrides pairs_per_cell

    def c(self):
        return _VhsParams(self.mass, self.sigma_v, self.T_scale, self.noise_sigma, self.shell_eps, self.d_ref,
                          self.omega, self.T_ref, self.pairs_per_cell, self.flags, self.cell_base,
                          _ptr(self.pairs_count, torch.int32) if self.pairs_count is not None else None)


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
    pairs_count: "torch.Tensor" = None  # device int32 [n_cells]: per-cell request, overrides pairs_per_cell

    def c(self):
        return _AbiParams(self.mass, self.b_max, self.lnE_min, self.lnE_max, self.chi_mode, self.pairs_per_cell,
                          self.flags, self.cell_base,
                          _ptr(self.pairs_count, torch.int32) if self.pairs_count is not None else None)


@dataclass
class CouetteParams:
    """1-D Couette layout (Q30): walls at x = 0 (-u_wall) and x = L (+u_wall), Maxwell wall model."""
    L: float
    dt: float
    u_wall: float
    rt_wall: float
    accommodation: float
    n_cells: int
    ntc_coef: float = 0.0      # F_N dt / V_c; > 0: NTC candidate counts every step of couette_run
    sigma_cr_max: float = 0.0  # uniform (sigma c_r)max bound of the NTC count and acceptance

    def c(self):
        return _CouetteParams(self.L, self.dt, self.u_wall, self.rt_wall, self.accommodation, self.n_cells,
                              self.ntc_coef, self.sigma_cr_max)


class PairDump:
    """Optional debug outputs of a fused step (device tensors with n entries)."""

    def __init__(self, n, device, gprime=True):
        self.pair_i = torch.full((n,), -1, dtype=torch.int32, device=device)
        self.pair_j = torch.full((n,), -1, dtype=torch.int32, device=device)
        self.accepted = torch.zeros(n, dtype=torch.uint8, device=device)
        self.gprime = torch.zeros((n, 3), dtype=torch.float32, device=device) if gprime else None
        self.aux = torch.zeros(n, dtype=torch.float32, device=device)

    def c(self):
        return _PairDump(_ptr(self.pair_i), _ptr(self.pair_j), _ptr(self.accepted), _ptr(self.gprime),
                         _ptr(self.aux))


NOALLOC_MAX_PARTICLES, NOALLOC_MAX_CELLS = 1 << 20, 1 << 17


def noalloc_setup():
    """once-per-device set-up of the no-allocation entry point, for the CURRENT device (torch.cuda.current_device())"""
    _chk(_lib.dsmc_noalloc_setup(), "dsmc_noalloc_setup")


def bin_noalloc(cell, vx, vy, vz, n_cells: int, out, status=None):
    """dsmc_bin_noalloc: the cell sort with a fixed file-scope scratch array instead of a context; allocates nothing
    (so `out` = (vx_s, vy_s, vz_s, perm, cell_start) must be given).  status: optional int32 device tensor [1].
    Enqueued on torch's current stream of the current device; calls that overlap on the GPU race on the scratch."""
    vx_s, vy_s, vz_s, perm, cell_start = out
    _chk(_lib.dsmc_bin_noalloc(C.c_void_p(torch.cuda.current_stream().cuda_stream), C.c_int64(cell.shape[0]),
                               C.c_int32(n_cells), _ptr(cell, torch.int32), _ptr(vx, torch.float32),
                               _ptr(vy, torch.float32), _ptr(vz, torch.float32), _ptr(vx_s), _ptr(vy_s), _ptr(vz_s),
                               _ptr(perm), _ptr(cell_start), _ptr(status, torch.int32) if status is not None else C.c_void_p(0)),
         "dsmc_bin_noalloc")
    return out


class Context:
    """dsmc_ctx wrapper.  Work is enqueued on torch's current stream at call time."""

    def __init__(self, max_particles: int, max_cells: int, device: int = 0):
        self._h = C.c_void_p()
        self.device = torch.device("cuda", device)
        _chk(_lib.dsmc_create(C.byref(self._h), C.c_int(device), C.c_int64(max_particles), C.c_int32(max_cells)),
             "dsmc_create")

    def close(self):
        if self._h:
            _lib.dsmc_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _stream(self):
        _chk(_lib.dsmc_set_stream(self._h, C.c_void_p(torch.cuda.current_stream(self.device).cuda_stream)),
             "dsmc_set_stream")

    def sync_status(self) -> int:
        return _lib.dsmc_sync_status(self._h)

    def check(self):
        _chk(self.sync_status(), "dsmc_sync_status")

    def launch_count(self) -> int:
        return int(_lib.dsmc_launch_count(self._h))

    # ---- operators
    def set_mlp(self, slot: int, weights, biases, act: int):
        L = len(weights)
        Ws = [np.ascontiguousarray(w, np.float32) for w in weights]
        bs = [np.ascontiguousarray(b, np.float32) for b in biases]
        d = _MlpDesc()
        d.n_layers = L
        d.act = act
        d.dims[0] = Ws[0].shape[1]
        for l in range(L):
            d.dims[l + 1] = Ws[l].shape[0]
        Wp = (C.POINTER(C.c_float) * L)(*[w.ctypes.data_as(C.POINTER(C.c_float)) for w in Ws])
        bp = (C.POINTER(C.c_float) * L)(*[b.ctypes.data_as(C.POINTER(C.c_float)) for b in bs])
        d.W, d.b = Wp, bp
        self._stream()
        _chk(_lib.dsmc_set_mlp(self._h, C.c_int(slot), C.byref(d)), "dsmc_set_mlp")

    def set_chi_table(self, chi: np.ndarray, lnE_min: float, lnE_max: float):
        chi = np.ascontiguousarray(chi, np.float32)
        self._stream()
        _chk(_lib.dsmc_set_chi_table(self._h, chi.ctypes.data_as(C.POINTER(C.c_float)), C.c_int32(chi.shape[0]),
                                     C.c_int32(chi.shape[1]), C.c_float(lnE_min), C.c_float(lnE_max)),
             "dsmc_set_chi_table")

    # ---- a1
    def bin(self, cell, vx, vy, vz, n_cells: int, out=None):
        n = cell.shape[0]
        dev = cell.device
        if out is None:
            out = (torch.empty(n, dtype=torch.float32, device=dev), torch.empty(n, dtype=torch.float32, device=dev),
                   torch.empty(n, dtype=torch.float32, device=dev), torch.empty(n, dtype=torch.int32, device=dev),
                   torch.empty(n_cells + 1, dtype=torch.int32, device=dev))
        vx_s, vy_s, vz_s, perm, cell_start = out
        self._stream()
        _chk(_lib.dsmc_bin(self._h, C.c_int64(n), C.c_int32(n_cells), _ptr(cell, torch.int32),
                           _ptr(vx, torch.float32), _ptr(vy, torch.float32), _ptr(vz, torch.float32),
                           _ptr(vx_s), _ptr(vy_s), _ptr(vz_s), _ptr(perm), _ptr(cell_start)), "dsmc_bin")
        return vx_s, vy_s, vz_s, perm, cell_start

    # ---- fused steps (in place on vx_s, vy_s, vz_s)
    def collide_vhs_nn(self, cell_start, vx_s, vy_s, vz_s, prm: VhsParams, seed: int, step: int,
                       sigma_cr_max=None, dump: PairDump = None):
        p = prm.c()
        d = dump.c() if dump is not None else None
        self._stream()
        _chk(_lib.dsmc_collide_vhs_nn(
            self._h, C.c_int64(vx_s.shape[0]), C.c_int32(cell_start.shape[0] - 1), _ptr(cell_start, torch.int32),
            _ptr(vx_s, torch.float32), _ptr(vy_s, torch.float32), _ptr(vz_s, torch.float32),
            _ptr(sigma_cr_max, torch.float32) if sigma_cr_max is not None else C.c_void_p(0), C.byref(p),
            C.c_uint64(seed), C.c_uint32(step), C.byref(d) if d is not None else None), "dsmc_collide_vhs_nn")

    def collide_abinitio(self, cell_start, vx_s, vy_s, vz_s, prm: AbinitioParams, seed: int, step: int,
                         cr_max=None, dump: PairDump = None):
        p = prm.c()
        d = dump.c() if dump is not None else None
        self._stream()
        _chk(_lib.dsmc_collide_abinitio(
            self._h, C.c_int64(vx_s.shape[0]), C.c_int32(cell_start.shape[0] - 1), _ptr(cell_start, torch.int32),
            _ptr(vx_s, torch.float32), _ptr(vy_s, torch.float32), _ptr(vz_s, torch.float32),
            _ptr(cr_max, torch.float32) if cr_max is not None else C.c_void_p(0), C.byref(p),
            C.c_uint64(seed), C.c_uint32(step), C.byref(d) if d is not None else None), "dsmc_collide_abinitio")

    # ---- moments
    def cell_moments(self, cell_start, vx_s, vy_s, vz_s, out=None):
        K = cell_start.shape[0] - 1
        if out is None:
            out = torch.empty((K, 4), dtype=torch.float64, device=cell_start.device)
        self._stream()
        _chk(_lib.dsmc_cell_moments(self._h, C.c_int64(vx_s.shape[0]), C.c_int32(K), _ptr(cell_start, torch.int32),
                                    _ptr(vx_s, torch.float32), _ptr(vy_s, torch.float32), _ptr(vz_s, torch.float32),
                                    _ptr(out, torch.float64)), "dsmc_cell_moments")
        return out

    def moment_match(self, cell_start, vx_s, vy_s, vz_s, target, flags: int = F_MOMENT_MATCH):
        self._stream()
        _chk(_lib.dsmc_moment_match(self._h, C.c_int64(vx_s.shape[0]), C.c_int32(cell_start.shape[0] - 1),
                                    _ptr(cell_start, torch.int32), _ptr(vx_s, torch.float32),
                                    _ptr(vy_s, torch.float32), _ptr(vz_s, torch.float32),
                                    _ptr(target, torch.float64), C.c_uint32(flags)), "dsmc_moment_match")

    # ---- a10
    def chi_batch(self, E_over_k, b, chi_mode: int, b_max: float, lnE_min=float(np.log(5.0)),
                  lnE_max=float(np.log(6.0e4)), flags: int = 0, out=None):
        if out is None:
            out = torch.empty_like(E_over_k)
        self._stream()
        _chk(_lib.dsmc_chi_batch(self._h, C.c_int64(E_over_k.shape[0]), _ptr(E_over_k, torch.float32),
                                 _ptr(b, torch.float32), _ptr(out, torch.float32), C.c_int32(chi_mode),
                                 C.c_float(b_max), C.c_float(lnE_min), C.c_float(lnE_max), C.c_uint32(flags)),
             "dsmc_chi_batch")
        return out

    def build_chi_table_lj(self, nE: int, nB: int, lnE_min=float(np.log(5.0)), lnE_max=float(np.log(6.0e4)),
                           b_max: float = 1e-9, eps_over_k: float = 119.8, sigma: float = 3.405e-10,
                           want_nodes: bool = False):
        """Generate the LJ chi table on the device and install it; returns the [nE, nB] node tensor if asked."""
        out = torch.empty((nE, nB), dtype=torch.float32, device=self.device) if want_nodes else None
        self._stream()
        _chk(_lib.dsmc_build_chi_table_lj(self._h, C.c_int32(nE), C.c_int32(nB), C.c_float(lnE_min), C.c_float(lnE_max),
                                          C.c_float(b_max), C.c_float(eps_over_k), C.c_float(sigma),
                                          _ptr(out, torch.float32) if out is not None else C.c_void_p(0)),
             "dsmc_build_chi_table_lj")
        return out

    def build_chi_table_mlp(self, nE: int, nB: int, lnE_min=float(np.log(5.0)), lnE_max=float(np.log(6.0e4)),
                            flags: int = 0, want_nodes: bool = False):
        """Generate the chi table on the device from the slot-1 chi-MLP and install it; flags 0 or F_BF16_TC."""
        out = torch.empty((nE, nB), dtype=torch.float32, device=self.device) if want_nodes else None
        self._stream()
        _chk(_lib.dsmc_build_chi_table_mlp(self._h, C.c_int32(nE), C.c_int32(nB), C.c_float(lnE_min), C.c_float(lnE_max),
                                           C.c_uint32(flags),
                                           _ptr(out, torch.float32) if out is not None else C.c_void_p(0)),
             "dsmc_build_chi_table_mlp")
        return out

    def chi_exact_batch(self, E_over_k, b, eps_over_k: float = 119.8, sigma: float = 3.405e-10, flags: int = 0,
                        out=None):
        """chi by the deflection-integral quadrature itself (LJ 12-6), signed unless flags & F_CHI_ABS."""
        if out is None:
            out = torch.empty_like(E_over_k)
        self._stream()
        _chk(_lib.dsmc_chi_exact_batch(self._h, C.c_int64(E_over_k.shape[0]), _ptr(E_over_k, torch.float32),
                                       _ptr(b, torch.float32), _ptr(out, torch.float32), C.c_float(eps_over_k),
                                       C.c_float(sigma), C.c_uint32(flags)), "dsmc_chi_exact_batch")
        return out

    # ---- f1: NTC candidate counts with carried remainder
    def ntc_counts(self, cell_start, sigma_cr_max, coef: float, remainder, out=None):
        """counts[k] = floor(1/2 N (N-1) coef sigma_cr_max[k] + remainder[k]); remainder (float64) updated in place."""
        K = cell_start.shape[0] - 1
        if out is None:
            out = torch.empty(K, dtype=torch.int32, device=cell_start.device)
        self._stream()
        _chk(_lib.dsmc_ntc_counts(self._h, C.c_int32(K), _ptr(cell_start, torch.int32),
                                  _ptr(sigma_cr_max, torch.float32), C.c_double(coef),
                                  _ptr(remainder, torch.float64), _ptr(out, torch.int32)), "dsmc_ntc_counts")
        return out

    # ---- f4: the minimal DSMC loop around the step (1-D Couette layout)
    def move_couette(self, x, vx, vy, vz, geo: "CouetteParams", seed: int, step: int, cell=None, bounces=None):
        """Free flight + Maxwell walls in place; returns the cell index array."""
        g = geo.c()
        if cell is None:
            cell = torch.empty(x.shape[0], dtype=torch.int32, device=x.device)
        self._stream()
        _chk(_lib.dsmc_move_couette(self._h, C.c_int64(x.shape[0]), _ptr(x, torch.float32), _ptr(vx, torch.float32),
                                    _ptr(vy, torch.float32), _ptr(vz, torch.float32), _ptr(cell, torch.int32),
                                    _ptr(bounces, torch.int32) if bounces is not None else C.c_void_p(0),
                                    C.byref(g), C.c_uint64(seed), C.c_uint32(step)), "dsmc_move_couette")
        return cell

    def gather_f32(self, perm, src, out=None):
        if out is None:
            out = torch.empty_like(src)
        self._stream()
        _chk(_lib.dsmc_gather_f32(self._h, C.c_int64(src.shape[0]), _ptr(perm, torch.int32),
                                  _ptr(src, torch.float32), _ptr(out, torch.float32)), "dsmc_gather_f32")
        return out

    def sample_cells(self, cell_start, vx_s, vy_s, vz_s, acc):
        self._stream()
        _chk(_lib.dsmc_sample_cells(self._h, C.c_int64(vx_s.shape[0]), C.c_int32(cell_start.shape[0] - 1),
                                    _ptr(cell_start, torch.int32), _ptr(vx_s, torch.float32),
                                    _ptr(vy_s, torch.float32), _ptr(vz_s, torch.float32),
                                    _ptr(acc, torch.float64)), "dsmc_sample_cells")
        return acc

    def couette_run(self, x, vx, vy, vz, geo: "CouetteParams", n_steps: int, vhs: VhsParams = None,
                    abi: AbinitioParams = None, seed: int = 0, step0: int = 0, sample_from: int = 0, acc=None):
        """n_steps of move -> bin -> gather -> collide -> sample on the device; x, v updated in place."""
        g = geo.c()
        pv = vhs.c() if vhs is not None else None
        pa = abi.c() if abi is not None else None
        self._stream()
        _chk(_lib.dsmc_couette_run(
            self._h, C.c_int64(x.shape[0]), _ptr(x, torch.float32), _ptr(vx, torch.float32),
            _ptr(vy, torch.float32), _ptr(vz, torch.float32), C.byref(g),
            C.byref(pv) if pv is not None else None, C.byref(pa) if pa is not None else None, C.c_uint64(seed),
            C.c_uint32(step0), C.c_int32(n_steps), C.c_int32(sample_from),
            _ptr(acc, torch.float64) if acc is not None else C.c_void_p(0)), "dsmc_couette_run")
        return acc

    # ---- end to end on host buffers (pinned CPU tensors)
    def step_host(self, cell_h, vx_h, vy_h, vz_h, n_cells, out_h, vhs: VhsParams = None,
                  abi: AbinitioParams = None, seed=0, step=0, submit_only=False):
        """out_h = (vx_out, vy_out, vz_out, perm, cell_start) CPU tensors.  Synchronous, unless submit_only: then the
        step is only enqueued (dsmc_step_host_submit) and the buffers belong to the library until sync_status()."""
        pv = vhs.c() if vhs is not None else None
        pa = abi.c() if abi is not None else None
        hp = lambda t: C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)
        self._stream()
        fn = _lib.dsmc_step_host_submit if submit_only else _lib.dsmc_step_host
        _chk(fn(
            self._h, C.c_int64(cell_h.shape[0]), C.c_int32(n_cells), hp(cell_h), hp(vx_h), hp(vy_h), hp(vz_h),
            hp(out_h[0]), hp(out_h[1]), hp(out_h[2]), hp(out_h[3]), hp(out_h[4]),
            C.byref(pv) if pv is not None else None, C.byref(pa) if pa is not None else None,
            C.c_uint64(seed), C.c_uint32(step)), "dsmc_step_host")
