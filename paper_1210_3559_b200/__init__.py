"""paper_1210_3559_b200 -- thin Python binding over libscmd (include/scmd.h).

Argument marshalling only: every step of the Sutton-Chen hot path (density sweep, force +
energy sweep, velocity-Verlet, thermostat) runs in the CUDA
kernels under csrc/.  PyTorch is used for device memory and streams.  There is no CPU
fallback: if libscmd.so is missing or no CUDA device is present, calls raise.
"""
from .distributed import RowSplitSuttonChen, row_range  # noqa: F401
from .binding import (  # noqa: F401
    SC_OK, SC_ERR_INVALID, SC_ERR_CUDA, SC_ERR_NOMEM, SC_ERR_STATE, SC_ERR_NONFINITE, SC_ERR_CAPACITY,
    SC_PREC_FP64, SC_PREC_MIXED, SC_THERMO_NONE, SC_THERMO_RESCALE, SC_THERMO_LANGEVIN,
    SC_OPT_ROWS_PER_THREAD, SC_OPT_LANES_PER_ROW, SC_OPT_WARPS_PER_CTA, SC_OPT_PERSISTENT,
    SC_OPT_ENERGY_EVERY_STEP, SC_OPT_NEIGHBOUR_CAPACITY, SC_OPT_LANGEVIN_STEP, SC_OPT_CELLS_PER_RADIUS,
    SC_OPT_ATOMS_PER_CTA, SC_OPT_NEWTON3, SC_OPT_CUTOFF_SHIFT, SC_OPT_NEWTON3_PIECES,
    SC_INFO_STEP_PATH, SC_INFO_NEIGHBOUR_CAPACITY, SC_INFO_NEIGHBOUR_CAPACITY_MAX, SC_INFO_ONE_LAUNCH, ScCreateOptions, load_probe_library,
    ScError, ScParams, ScThermostat, SuttonChen, load_library, library_path, exported_symbols,
    probe_throughput, probe_reciprocal, NI_PARAMS, rescale_thermostat, langevin_thermostat,
    sc_density_noalloc, SC_NOALLOC_MAX_ATOMS,
)
