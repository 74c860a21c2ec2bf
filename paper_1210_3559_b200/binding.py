"""ctypes binding of libscmd's C ABI (include/scmd.h): same names, marshalling only."""
from __future__ import annotations

import ctypes
import re
from pathlib import Path

PKG = Path(__file__).resolve().parent
_LIB_PATH = PKG / "libscmd.so"
_PROBE_LIB_PATH = PKG / "libscmd_probe.so"
_HEADER = PKG.parent / "include" / "scmd.h"
_PROBE_HEADER = PKG.parent / "include" / "scmd_probe.h"

SC_OK, SC_ERR_INVALID, SC_ERR_CUDA, SC_ERR_NOMEM, SC_ERR_STATE, SC_ERR_NONFINITE, SC_ERR_CAPACITY = range(7)
SC_PREC_FP64, SC_PREC_MIXED = 0, 1
SC_THERMO_NONE, SC_THERMO_RESCALE, SC_THERMO_LANGEVIN = 0, 1, 2
(SC_OPT_ROWS_PER_THREAD, SC_OPT_LANES_PER_ROW, SC_OPT_WARPS_PER_CTA, SC_OPT_PERSISTENT,
 SC_OPT_ENERGY_EVERY_STEP, SC_OPT_NEIGHBOUR_CAPACITY, SC_OPT_LANGEVIN_STEP, SC_OPT_CELLS_PER_RADIUS,
 SC_OPT_ATOMS_PER_CTA, SC_OPT_NEWTON3, SC_OPT_CUTOFF_SHIFT, SC_OPT_NEWTON3_PIECES) = range(1, 13)
SC_INFO_STEP_PATH, SC_INFO_NEIGHBOUR_CAPACITY, SC_INFO_NEIGHBOUR_CAPACITY_MAX, SC_INFO_ONE_LAUNCH = 100, 101, 102, 103
_STATUS_NAMES = ["SC_OK", "SC_ERR_INVALID", "SC_ERR_CUDA", "SC_ERR_NOMEM", "SC_ERR_STATE",
                 "SC_ERR_NONFINITE", "SC_ERR_CAPACITY"]

# Sutton-Chen nickel; mass from BASELINE.json
NI_PARAMS = dict(n=9, m=6, eps=1.5707e-2, c=39.432, a=3.52, mass=58.69)


class ScParams(ctypes.Structure):
    _fields_ = [("n", ctypes.c_int32), ("m", ctypes.c_int32), ("eps", ctypes.c_double),
                ("c", ctypes.c_double), ("a", ctypes.c_double), ("mass", ctypes.c_double),
                ("r_cut", ctypes.c_double)]


class ScCreateOptions(ctypes.Structure):
    _fields_ = [("neighbour_capacity", ctypes.c_int32), ("newton3_storage", ctypes.c_int32),
                ("row_begin", ctypes.c_int32), ("row_end", ctypes.c_int32), ("reserved", ctypes.c_int32 * 4)]


class ScThermostat(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_int32), ("T_start", ctypes.c_double), ("T_end", ctypes.c_double),
                ("gamma", ctypes.c_double), ("seed", ctypes.c_uint64)]


class ScError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        self.status = status
        name = _STATUS_NAMES[status] if 0 <= status < len(_STATUS_NAMES) else str(status)
        super().__init__(f"{where}: {name}" + (f" ({detail})" if detail else ""))


_lib = None


def library_path() -> Path:
    return _LIB_PATH


def exported_symbols(header: Path | None = None) -> list[str]:
    """Function names include/scmd.h (or the given header) declares (parsed from the header)."""
    text = (header or _HEADER).read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sc_[a-z_0-9]+)\s*\(", text)))


def load_library() -> ctypes.CDLL:
    """dlopen libscmd.so (built in-tree by paper_1210_3559_b200/build.py).  Raises if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not _LIB_PATH.exists():
        raise ScError(SC_ERR_CUDA, "load_library",
                      f"{_LIB_PATH} not found: run `python -c 'import __graft_entry__ as g; g.build()'`")
    L = ctypes.CDLL(str(_LIB_PATH))
    vp, i32, i64, dbl, sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_double, ctypes.c_size_t
    PP, TP = ctypes.POINTER(ScParams), ctypes.POINTER(ScThermostat)
    DP, IP = ctypes.POINTER(dbl), ctypes.POINTER(i64)
    sig = {
        "sc_workspace_bytes": (sz, [PP, i64, i32, dbl]),
        "sc_workspace_bytes_ex": (sz, [PP, i64, i32, dbl, ctypes.POINTER(ScCreateOptions)]),
        "sc_create": (i32, [PP, i64, i32, dbl, vp, sz, vp, ctypes.POINTER(vp)]),
        "sc_create_ex": (i32, [PP, i64, i32, dbl, ctypes.POINTER(ScCreateOptions), vp, sz, vp, ctypes.POINTER(vp)]),
        "sc_destroy": (i32, [vp]),
        "sc_set_option": (i32, [vp, i32, i64]),
        "sc_get_option": (i32, [vp, i32, IP]),
        "sc_set_state": (i32, [vp, vp, vp]),
        "sc_get_state": (i32, [vp, vp, vp]),
        "sc_density": (i32, [vp, vp]),
        "sc_forces": (i32, [vp, vp]),
        "sc_energy": (i32, [vp, DP]),
        "sc_kinetic": (i32, [vp, DP, DP]),
        "sc_step": (i32, [vp, dbl, TP, i64]),
        "sc_step_rows": (i32, [vp, i32, dbl, TP, vp, vp]),
        "sc_stats": (i32, [vp, IP, IP, IP]),
        "sc_eval_host": (i32, [vp, vp, vp, vp, DP]),
        "sc_step_host": (i32, [vp, vp, vp, dbl, TP, i64, DP]),
        "sc_rdf": (i32, [vp, DP, dbl, dbl, i32, IP, IP, DP]),
        "sc_msd": (i32, [vp, vp, dbl, i32, DP, IP, DP]),
        "sc_launch_count": (i32, [vp, IP]),
        "sc_profile": (i32, [vp, i32]),
        "sc_profile_read": (i32, [vp, DP, DP]),
        "sc_last_error": (ctypes.c_char_p, [vp]),
        "sc_version": (ctypes.c_char_p, []),
        "sc_density_noalloc": (i32, [PP, i64, vp, vp, vp, vp]),
        "sc_noalloc_last_error": (ctypes.c_char_p, []),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype, fn.argtypes = res, args
    _lib = L
    return L


_probe_lib = None


def load_probe_library() -> ctypes.CDLL:
    """dlopen libscmd_probe.so (include/scmd_probe.h): diagnostics for bench.py and the tests, not the product."""
    global _probe_lib
    if _probe_lib is not None:
        return _probe_lib
    if not _PROBE_LIB_PATH.exists():
        raise ScError(SC_ERR_CUDA, "load_probe_library", f"{_PROBE_LIB_PATH} not found: run __graft_entry__.build()")
    L = ctypes.CDLL(str(_PROBE_LIB_PATH))
    vp, i32, dbl, sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_double, ctypes.c_size_t
    DP = ctypes.POINTER(dbl)
    L.sc_probe_throughput.restype, L.sc_probe_throughput.argtypes = i32, [i32, vp, vp, sz, DP, DP]
    L.sc_probe_reciprocal.restype, L.sc_probe_reciprocal.argtypes = i32, [dbl, dbl, i32, vp, vp, sz, DP]
    _probe_lib = L
    return L


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise ScError(SC_ERR_CUDA, "libscmd", "no CUDA device: the Sutton-Chen path has no CPU fallback")
    return torch


def _dev_ptr(t, n_elems: int, what: str) -> int:
    torch = _torch()
    if t is None:
        return 0
    if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == n_elems):
        raise ScError(SC_ERR_INVALID, what, f"need a contiguous CUDA float64 tensor of {n_elems} elements")
    return t.data_ptr()


def _host_ptr(a, n_elems: int, what: str) -> int:
    import numpy as np
    torch = _torch()
    if a is None:
        return 0
    if isinstance(a, torch.Tensor):
        if a.is_cuda or a.dtype != torch.float64 or not a.is_contiguous() or a.numel() != n_elems:
            raise ScError(SC_ERR_INVALID, what, f"need a contiguous CPU float64 tensor of {n_elems} elements")
        return a.data_ptr()
    if not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous and a.size == n_elems):
        raise ScError(SC_ERR_INVALID, what, f"need a contiguous float64 array of {n_elems} elements")
    return a.ctypes.data


class SuttonChen:
    """One libscmd context: owns a torch workspace tensor and the opaque sc_ctx."""

    def __init__(self, n_atoms: int, *, n=9, m=6, eps=1.5707e-2, c=39.432, a=3.52, mass=58.69, r_cut=0.0,
                 precision: int = SC_PREC_FP64, skin: float = 0.0, device=None, stream=None, poison: bool = False,
                 neighbour_capacity: int = 0, newton3_storage: int = 0, row_begin: int = 0, row_end: int = 0):
        torch = _torch()
        self.lib = load_library()
        self.n_atoms = int(n_atoms)
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        self.params = ScParams(int(n), int(m), float(eps), float(c), float(a), float(mass), float(r_cut))
        self.precision = int(precision)
        self._ctx = ctypes.c_void_p()
        opts = ScCreateOptions(int(neighbour_capacity), int(newton3_storage), int(row_begin), int(row_end))
        with torch.cuda.device(self.device):
            nbytes = self.lib.sc_workspace_bytes_ex(ctypes.byref(self.params), self.n_atoms, self.precision, float(skin),
                                                    ctypes.byref(opts))
            if nbytes == 0:
                raise ScError(SC_ERR_INVALID, "sc_workspace_bytes", "invalid parameters")
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            if poison:                       # every byte 0xFF (NaN as binary64 / binary32, -1 as int): the library must
                self.workspace.fill_(255)    # never read workspace memory it has not written itself
            base = (self.workspace.data_ptr() + 255) // 256 * 256
            self.stream = torch.cuda.current_stream(self.device) if stream is None else stream
            st = self.lib.sc_create_ex(ctypes.byref(self.params), self.n_atoms, self.precision, float(skin),
                                       ctypes.byref(opts), base, nbytes, self.stream.cuda_stream, ctypes.byref(self._ctx))
        if st != SC_OK:
            self._ctx = ctypes.c_void_p()
            raise ScError(st, "sc_create")

    # -- plumbing ----------------------------------------------------------------------------
    def _check(self, st: int, where: str):
        if st != SC_OK:
            msg = self.lib.sc_last_error(self._ctx)
            raise ScError(st, where, msg.decode() if msg else "")

    def close(self):
        if getattr(self, "_ctx", None) and self._ctx.value:
            self.lib.sc_destroy(self._ctx)
            self._ctx = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _new(self, *shape):
        return _torch().empty(*shape, dtype=_torch().float64, device=self.device)

    # -- the C ABI, name for name ------------------------------------------------------------
    def sc_set_option(self, option: int, value: int):
        self._check(self.lib.sc_set_option(self._ctx, int(option), int(value)), "sc_set_option")

    def sc_get_option(self, option: int) -> int:
        v = ctypes.c_int64()
        self._check(self.lib.sc_get_option(self._ctx, int(option), ctypes.byref(v)), "sc_get_option")
        return v.value

    def sc_set_state(self, d_pos, d_vel=None):
        n3 = 3 * self.n_atoms
        self._check(self.lib.sc_set_state(self._ctx, _dev_ptr(d_pos, n3, "d_pos"), _dev_ptr(d_vel, n3, "d_vel")),
                    "sc_set_state")

    def sc_get_state(self, want_vel: bool = True):
        pos = self._new(self.n_atoms, 3)
        vel = self._new(self.n_atoms, 3) if want_vel else None
        self._check(self.lib.sc_get_state(self._ctx, pos.data_ptr(), vel.data_ptr() if want_vel else 0), "sc_get_state")
        return pos, vel

    def sc_density(self, out=None):
        rho = self._new(self.n_atoms) if out is None else out
        self._check(self.lib.sc_density(self._ctx, _dev_ptr(rho, self.n_atoms, "d_rho")), "sc_density")
        return rho

    def sc_forces(self, out=None):
        f = self._new(self.n_atoms, 3) if out is None else out
        self._check(self.lib.sc_forces(self._ctx, _dev_ptr(f, 3 * self.n_atoms, "d_force")), "sc_forces")
        return f

    def sc_energy(self) -> float:
        e = ctypes.c_double()
        self._check(self.lib.sc_energy(self._ctx, ctypes.byref(e)), "sc_energy")
        return e.value

    def sc_kinetic(self):
        ke, t = ctypes.c_double(), ctypes.c_double()
        self._check(self.lib.sc_kinetic(self._ctx, ctypes.byref(ke), ctypes.byref(t)), "sc_kinetic")
        return ke.value, t.value

    def sc_step(self, dt_fs: float, nsteps: int, thermostat: ScThermostat | None = None):
        th = ctypes.byref(thermostat) if thermostat is not None else None
        self._check(self.lib.sc_step(self._ctx, float(dt_fs), th, int(nsteps)), "sc_step")

    def sc_step_rows(self, phase: int, dt_fs: float, d_pos_all, d_rho_all, thermostat: ScThermostat | None = None):
        """One phase of a row-split step (include/scmd.h): d_pos_all [>= N*3], d_rho_all [>= N] are the caller's
        all-atoms device arrays (they may be longer: padded for equal all-gather chunks)."""
        torch = _torch()
        for t_, n_ in ((d_pos_all, 3 * self.n_atoms), (d_rho_all, self.n_atoms)):
            if t_ is not None and not (t_.is_cuda and t_.dtype == torch.float64 and t_.is_contiguous() and t_.numel() >= n_):
                raise ScError(SC_ERR_INVALID, "sc_step_rows", f"need a contiguous CUDA float64 tensor of >= {n_} elements")
        th = ctypes.byref(thermostat) if thermostat is not None else None
        self._check(self.lib.sc_step_rows(self._ctx, int(phase), float(dt_fs), th,
                                          0 if d_pos_all is None else d_pos_all.data_ptr(),
                                          0 if d_rho_all is None else d_rho_all.data_ptr()), "sc_step_rows")

    def sc_stats(self):
        a, b, c = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64()
        self._check(self.lib.sc_stats(self._ctx, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)), "sc_stats")
        return dict(n_rebuilds=a.value, n_pairs_in_cut=b.value, max_neighbours=c.value)

    def sc_eval_host(self, h_pos, h_force=None, h_rho=None) -> float:
        n = self.n_atoms
        e = ctypes.c_double()
        self._check(self.lib.sc_eval_host(self._ctx, _host_ptr(h_pos, 3 * n, "h_pos"), _host_ptr(h_force, 3 * n, "h_force"),
                                          _host_ptr(h_rho, n, "h_rho"), ctypes.byref(e)), "sc_eval_host")
        return e.value

    def sc_step_host(self, h_pos, h_vel, dt_fs: float, nsteps: int, thermostat: ScThermostat | None = None):
        n3 = 3 * self.n_atoms
        s = (ctypes.c_double * 3)()
        th = ctypes.byref(thermostat) if thermostat is not None else None
        self._check(self.lib.sc_step_host(self._ctx, _host_ptr(h_pos, n3, "h_pos"), _host_ptr(h_vel, n3, "h_vel"),
                                          float(dt_fs), th, int(nsteps), s), "sc_step_host")
        return dict(epot=s[0], ekin=s[1], temperature=s[2])

    def sc_rdf(self, r_select: float, bin_width: float, n_bins: int, centre=None):
        """-> (counts[n_bins] numpy int64, n_ref, centre used); see sc_rdf in include/scmd.h."""
        import numpy as np
        counts = np.zeros(int(n_bins), dtype=np.int64)
        n_ref = ctypes.c_int64()
        used = (ctypes.c_double * 3)()
        cen = None
        if centre is not None:
            cen = (ctypes.c_double * 3)(*[float(v) for v in centre])
        self._check(self.lib.sc_rdf(self._ctx, cen, float(r_select), float(bin_width), int(n_bins),
                                    counts.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)), ctypes.byref(n_ref), used),
                    "sc_rdf")
        return counts, n_ref.value, np.array(list(used))

    def sc_msd(self, ref_pos, r_centre: float = 0.0, align: int = 2):
        """-> (msd in A^2, n_sel, R[3,3] numpy); ref_pos: device tensor [N,3] float64; see sc_msd in include/scmd.h."""
        import numpy as np
        msd, n_sel = ctypes.c_double(), ctypes.c_int64()
        rot = (ctypes.c_double * 9)()
        self._check(self.lib.sc_msd(self._ctx, _dev_ptr(ref_pos, 3 * self.n_atoms, "d_ref_pos"), float(r_centre), int(align),
                                    ctypes.byref(msd), ctypes.byref(n_sel), rot), "sc_msd")
        return msd.value, n_sel.value, np.array(list(rot)).reshape(3, 3)

    def sc_launch_count(self) -> int:
        v = ctypes.c_int64()
        self._check(self.lib.sc_launch_count(self._ctx, ctypes.byref(v)), "sc_launch_count")
        return v.value

    def sc_profile(self, enable: bool):
        self._check(self.lib.sc_profile(self._ctx, 1 if enable else 0), "sc_profile")

    def sc_profile_read(self):
        a, b = ctypes.c_double(), ctypes.c_double()
        self._check(self.lib.sc_profile_read(self._ctx, ctypes.byref(a), ctypes.byref(b)), "sc_profile_read")
        return dict(ms_density=a.value, ms_force=b.value)


SC_NOALLOC_MAX_ATOMS = 16384


def sc_density_noalloc(d_pos, d_rho, d_sum_sqrt_rho=None, *, n=9, m=6, eps=1.5707e-2, c=39.432, a=3.52, mass=58.69,
                       stream=None) -> None:
    """include/scmd.h sc_density_noalloc: rho_i (all pairs, FP64) into the caller's `d_rho` and sum_i sqrt(rho_i) into
    the caller's one-element `d_sum_sqrt_rho`, with the library's scratch in a static device array: no workspace, no
    allocation inside the call (the tensors passed in are the caller's).  N <= SC_NOALLOC_MAX_ATOMS."""
    torch = _torch()
    lib = load_library()
    if not (d_pos.is_cuda and d_rho.is_cuda and d_pos.dtype == torch.float64 and d_rho.dtype == torch.float64
            and d_pos.is_contiguous() and d_rho.is_contiguous() and d_pos.dim() == 2 and d_pos.shape[1] == 3
            and d_rho.numel() == d_pos.shape[0]):
        raise ScError(SC_ERR_INVALID, "sc_density_noalloc", "need contiguous float64 CUDA tensors pos[N, 3], rho[N]")
    if d_sum_sqrt_rho is not None and not (d_sum_sqrt_rho.is_cuda and d_sum_sqrt_rho.dtype == torch.float64
                                           and d_sum_sqrt_rho.numel() == 1):
        raise ScError(SC_ERR_INVALID, "sc_density_noalloc", "sum_sqrt_rho must be a one-element float64 CUDA tensor")
    params = ScParams(int(n), int(m), float(eps), float(c), float(a), float(mass), 0.0)
    with torch.cuda.device(d_pos.device):
        s = torch.cuda.current_stream(d_pos.device) if stream is None else stream
        st = lib.sc_density_noalloc(ctypes.byref(params), int(d_pos.shape[0]), d_pos.data_ptr(), d_rho.data_ptr(),
                                    d_sum_sqrt_rho.data_ptr() if d_sum_sqrt_rho is not None else None, s.cuda_stream)
    if st != SC_OK:
        msg = lib.sc_noalloc_last_error()
        raise ScError(st, "sc_density_noalloc", msg.decode() if msg else "")


def rescale_thermostat(T_start: float, T_end: float) -> ScThermostat:
    return ScThermostat(SC_THERMO_RESCALE, float(T_start), float(T_end), 0.0, 0)


def langevin_thermostat(T_start: float, T_end: float, gamma_per_fs: float, seed: int) -> ScThermostat:
    return ScThermostat(SC_THERMO_LANGEVIN, float(T_start), float(T_end), float(gamma_per_fs), int(seed))


def probe_throughput(kind: int):
    """-> (thread-level instructions per second, SM clock MHz); see sc_probe_throughput."""
    torch = _torch()
    L = load_probe_library()
    scratch = torch.zeros(1 << 16, dtype=torch.uint8, device="cuda")
    v, mhz = ctypes.c_double(), ctypes.c_double()
    st = L.sc_probe_throughput(int(kind), torch.cuda.current_stream().cuda_stream, scratch.data_ptr(), scratch.numel(),
                               ctypes.byref(v), ctypes.byref(mhz))
    if st != SC_OK:
        raise ScError(st, "sc_probe_throughput")
    return v.value, mhz.value


def probe_reciprocal(lo: float, hi: float, n_samples: int = 1 << 22):
    """-> dict of maximum relative errors of the FP64 reciprocal building blocks."""
    torch = _torch()
    L = load_probe_library()
    scratch = torch.zeros(1 << 16, dtype=torch.uint8, device="cuda")
    out = (ctypes.c_double * 4)()
    st = L.sc_probe_reciprocal(float(lo), float(hi), int(n_samples), torch.cuda.current_stream().cuda_stream,
                               scratch.data_ptr(), scratch.numel(), out)
    if st != SC_OK:
        raise ScError(st, "sc_probe_reciprocal")
    return dict(rcp_seed=out[0], rcp=out[1], rsqrt_seed=out[2], rsqrt=out[3])
