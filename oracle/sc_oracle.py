"""ctypes wrapper around oracle/sc_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this.  It never imports the CUDA package.  See sc_oracle.c's header
for what is computed and which passage of PAPER.md each function follows.

Two shared objects are built from the one C file:
  liboracle_ld.so              long-double pair arithmetic + accumulators  (parity reference; gcc -O2)
  liboracle_plain_<host>.so    binary64 throughout (the timed baseline; gcc -O3 -march=native -fopenmp as SURVEY.md
                               section 8(d) prescribes, still no fast-math and no FMA contraction).  -march=native code
                               must not travel between machines, so the file name carries a hash of this host's CPU
                               flags and compiler version: the GPU box builds its own copy on first use.
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import platform
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "sc_oracle.c"


def _host_tag() -> str:
    """Short hash of what -march=native depends on: the CPU feature flags and the compiler version."""
    flags = platform.machine()
    try:
        for line in Path("/proc/cpuinfo").read_text().splitlines():
            if line.startswith(("flags", "Features")):
                flags += line
                break
    except OSError:
        pass
    try:
        flags += subprocess.run(["gcc", "-dumpfullversion"], capture_output=True, text=True).stdout
    except OSError:
        pass
    return hashlib.sha1(flags.encode()).hexdigest()[:10]


_VARIANTS = {
    "ld": (_HERE / "liboracle_ld.so", ["-O2", "-DSC_ORACLE_LONG_DOUBLE"]),
    "plain": (_HERE / f"liboracle_plain_{_host_tag()}.so", ["-O3", "-march=native"]),
}


class OracleParams(ctypes.Structure):
    _fields_ = [("n", ctypes.c_int32), ("m", ctypes.c_int32),
                ("eps", ctypes.c_double), ("c", ctypes.c_double), ("a", ctypes.c_double),
                ("mass", ctypes.c_double), ("r_cut", ctypes.c_double), ("cut_shift", ctypes.c_int32)]


def build(force: bool = False) -> None:
    """Compile both variants with gcc (no fast-math, no FMA contraction)."""
    for name, (so, defs) in _VARIANTS.items():
        if not force and so.exists() and so.stat().st_mtime >= _SRC.stat().st_mtime:
            continue
        cmd = ["gcc", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               "-fno-fast-math", *defs, str(_SRC), "-o", str(so), "-lm"]
        subprocess.run(cmd, check=True)


_DP = ctypes.POINTER(ctypes.c_double)
_IP = ctypes.POINTER(ctypes.c_int64)


def _dptr(a):
    return None if a is None else a.ctypes.data_as(_DP)


class Oracle:
    """One loaded variant of the C oracle."""

    def __init__(self, variant: str = "ld"):
        build()
        so, _ = _VARIANTS[variant]
        self.variant = variant
        self.lib = ctypes.CDLL(str(so))
        L = self.lib
        PP = ctypes.POINTER(OracleParams)
        L.oracle_real_bits.restype = ctypes.c_int
        L.oracle_density.argtypes = [ctypes.c_int64, _DP, PP, _DP]
        L.oracle_energy_forces.argtypes = [ctypes.c_int64, _DP, PP, _DP, _DP, _DP]
        L.oracle_forces_rows.argtypes = [ctypes.c_int64, _DP, PP, _DP, _IP, ctypes.c_int64, _DP, _DP]
        L.oracle_density_rows.argtypes = [ctypes.c_int64, _DP, PP, _IP, ctypes.c_int64, _DP]
        L.oracle_kinetic.argtypes = [ctypes.c_int64, _DP, ctypes.c_double, _DP, _DP]
        L.oracle_count_pairs.argtypes = [ctypes.c_int64, _DP, ctypes.c_double]
        L.oracle_count_pairs.restype = ctypes.c_int64
        L.oracle_run.argtypes = [ctypes.c_int64, _DP, _DP, PP, ctypes.c_double, ctypes.c_int64,
                                 ctypes.c_int32, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                 ctypes.c_uint64, ctypes.c_uint64, _DP, _DP, _DP]
        L.oracle_rdf_counts.argtypes = [ctypes.c_int64, _DP, _DP, ctypes.c_double, ctypes.c_double, ctypes.c_int64, _IP, _DP]
        L.oracle_rdf_counts.restype = ctypes.c_int64
        U32P = ctypes.POINTER(ctypes.c_uint32)
        L.oracle_philox4x32_10.argtypes = [U32P, U32P, U32P]
        L.oracle_philox4x32_10.restype = None
        L.oracle_langevin_normals.argtypes = [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint64, _DP]
        L.oracle_langevin_normals.restype = None

    @staticmethod
    def params(n=9, m=6, eps=1.5707e-2, c=39.432, a=3.52, mass=58.69, r_cut=0.0, cut_shift=0) -> OracleParams:
        return OracleParams(int(n), int(m), float(eps), float(c), float(a), float(mass), float(r_cut), int(cut_shift))

    @staticmethod
    def _pos(pos) -> np.ndarray:
        p = np.ascontiguousarray(pos, dtype=np.float64)
        assert p.ndim == 2 and p.shape[1] == 3
        return p

    def density(self, pos, params: OracleParams) -> np.ndarray:
        p = self._pos(pos)
        rho = np.zeros(p.shape[0], dtype=np.float64)
        rc = self.lib.oracle_density(p.shape[0], _dptr(p), ctypes.byref(params), _dptr(rho))
        assert rc == 0
        return rho

    def energy_forces(self, pos, params: OracleParams):
        """-> (rho[N], F[N,3], (U, U_pair, U_emb))"""
        p = self._pos(pos)
        n = p.shape[0]
        rho = np.zeros(n, dtype=np.float64)
        f = np.zeros((n, 3), dtype=np.float64)
        e = np.zeros(3, dtype=np.float64)
        rc = self.lib.oracle_energy_forces(n, _dptr(p), ctypes.byref(params), _dptr(rho), _dptr(f), _dptr(e))
        assert rc == 0
        return rho, f, (float(e[0]), float(e[1]), float(e[2]))

    def energy(self, pos, params: OracleParams) -> float:
        return self.energy_forces(pos, params)[2][0]

    def forces_rows(self, pos, params: OracleParams, rho_all, rows):
        p = self._pos(pos)
        rows = np.ascontiguousarray(rows, dtype=np.int64)
        rho_all = np.ascontiguousarray(rho_all, dtype=np.float64)
        f = np.zeros((rows.size, 3), dtype=np.float64)
        ps = np.zeros(rows.size, dtype=np.float64)
        rc = self.lib.oracle_forces_rows(p.shape[0], _dptr(p), ctypes.byref(params), _dptr(rho_all),
                                         rows.ctypes.data_as(_IP), rows.size, _dptr(f), _dptr(ps))
        assert rc == 0
        return f, ps

    def density_rows(self, pos, params: OracleParams, rows) -> np.ndarray:
        p = self._pos(pos)
        rows = np.ascontiguousarray(rows, dtype=np.int64)
        rho = np.zeros(rows.size, dtype=np.float64)
        rc = self.lib.oracle_density_rows(p.shape[0], _dptr(p), ctypes.byref(params),
                                          rows.ctypes.data_as(_IP), rows.size, _dptr(rho))
        assert rc == 0
        return rho

    def kinetic(self, vel, mass: float = 58.69):
        v = np.ascontiguousarray(vel, dtype=np.float64)
        ke = ctypes.c_double(); t = ctypes.c_double()
        rc = self.lib.oracle_kinetic(v.shape[0], _dptr(v), float(mass), ctypes.byref(ke), ctypes.byref(t))
        assert rc == 0
        return ke.value, t.value

    def count_pairs(self, pos, r_cut: float) -> int:
        p = self._pos(pos)
        return int(self.lib.oracle_count_pairs(p.shape[0], _dptr(p), float(r_cut)))

    def rdf_counts(self, pos, r_select: float, bin_width: float, n_bins: int, centre=None):
        """-> (counts[n_bins] int64, n_ref, centre used)."""
        p = self._pos(pos)
        counts = np.zeros(int(n_bins), dtype=np.int64)
        cen = None if centre is None else np.ascontiguousarray(centre, dtype=np.float64)
        out = np.zeros(3)
        n_ref = self.lib.oracle_rdf_counts(p.shape[0], _dptr(p), _dptr(cen), float(r_select), float(bin_width),
                                           int(n_bins), counts.ctypes.data_as(_IP), _dptr(out))
        return counts, int(n_ref), out

    @staticmethod
    def msd_aligned(pos, ref, r_centre: float = 0.0, align: int = 2):
        """Mean-square displacement of Eq. (12)'s numerator after the rigid-body fit of
        PAPER.md:209: "cluster was translated and rotated as a whole in order to minimize the root-mean-square
        displacement of atoms from a reference structure ... the diffusion coefficient was calculated for all
        atoms located within 10 A of the cluster center of mass".  Plain numpy in binary64, written out as the
        definition: centroids (equal masses), the proper rotation that minimises sum_i |R x_i' - y_i'|^2 over
        ALL atoms (Kabsch: SVD of the 3x3 covariance, det fixed to +1), then the mean of |R x_i' - y_i'|^2 over
        the atoms whose REFERENCE position lies strictly within r_centre of the reference centroid (DESIGN.md
        Q20; r_centre <= 0: every atom).  align: 0 none, 1 translation only, 2 translation + rotation.
        -> (msd in A^2, number of selected atoms, R[3,3]); msd = 0.0 when nothing is selected."""
        x = np.ascontiguousarray(pos, dtype=np.float64).reshape(-1, 3)
        y = np.ascontiguousarray(ref, dtype=np.float64).reshape(-1, 3)
        assert x.shape == y.shape
        cy = y.mean(axis=0)
        yc = y - cy
        if align == 0:
            xc = x - cy                       # no fit: plain displacement y_i - x_i, selection about the reference centroid
        else:
            xc = x - x.mean(axis=0)
        R = np.eye(3)
        if align == 2:
            H = xc.T @ yc                     # H_ab = sum_i x'_ia y'_ib
            U, _, Vt = np.linalg.svd(H)
            d = 1.0 if np.linalg.det(Vt.T @ U.T) >= 0.0 else -1.0
            R = Vt.T @ np.diag([1.0, 1.0, d]) @ U.T
        disp2 = ((xc @ R.T - yc) ** 2).sum(axis=1)
        sel = np.ones(len(y), dtype=bool) if not (r_centre > 0.0) else (yc ** 2).sum(axis=1) < r_centre ** 2
        n_sel = int(sel.sum())
        return (float(disp2[sel].mean()) if n_sel else 0.0), n_sel, R

    def philox4x32_10(self, ctr, key) -> np.ndarray:
        c = np.ascontiguousarray(ctr, dtype=np.uint32); k = np.ascontiguousarray(key, dtype=np.uint32)
        out = np.zeros(4, dtype=np.uint32)
        U32P = ctypes.POINTER(ctypes.c_uint32)
        self.lib.oracle_philox4x32_10(c.ctypes.data_as(U32P), k.ctypes.data_as(U32P), out.ctypes.data_as(U32P))
        return out

    def langevin_normals(self, seed: int, atom: int, step: int) -> np.ndarray:
        xi = np.zeros(3)
        self.lib.oracle_langevin_normals(int(seed), int(atom), int(step), _dptr(xi))
        return xi

    def run(self, pos, vel, params: OracleParams, dt: float, nsteps: int, thermo_kind: int = 0,
            T_start: float = 0.0, T_end: float = 0.0, traces: bool = True, pos_trace: bool = False,
            gamma: float = 0.0, seed: int = 0, step0: int = 0):
        """-> dict(pos, vel, epot[nsteps+1], ekin[nsteps+1], pos_trace or None)"""
        p = self._pos(pos).copy()
        v = np.ascontiguousarray(vel, dtype=np.float64).copy()
        n = p.shape[0]
        ep = np.zeros(nsteps + 1) if traces else None
        ek = np.zeros(nsteps + 1) if traces else None
        pt = np.zeros((nsteps + 1, n, 3)) if pos_trace else None
        rc = self.lib.oracle_run(n, _dptr(p), _dptr(v), ctypes.byref(params), float(dt), int(nsteps),
                                 int(thermo_kind), float(T_start), float(T_end), float(gamma), int(seed), int(step0),
                                 _dptr(ep), _dptr(ek), _dptr(pt))
        assert rc == 0
        return dict(pos=p, vel=v, epot=ep, ekin=ek, pos_trace=pt)


def set_threads(n: int) -> None:
    """OpenMP thread count for subsequent calls (env var is read at first parallel region
    only, so go through the runtime)."""
    for so, _ in _VARIANTS.values():
        if so.exists():
            try:
                omp = ctypes.CDLL("libgomp.so.1")
                omp.omp_set_num_threads(int(n))
                return
            except OSError:
                os.environ["OMP_NUM_THREADS"] = str(int(n))
                return
