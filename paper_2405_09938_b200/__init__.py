"""B200-native hot path of the HEEPS/MARE raw-data generator (arXiv 2405.09938).

Thin Python binding over the C ABI in include/heeps_sim.h: argument marshalling only --
every step of the path (kinematics, geometry/gains/amplitude/cull, echo accumulation,
finalize) runs in the hand-written CUDA kernels of `csrc/`.  PyTorch is used for device
memory and streams.  There is no CPU fallback: importing `binding` without the built
library, or creating a simulator without a CUDA device, fails loudly.
"""
from .binding import (  # noqa: F401
    LIBRARY_PATH,
    SimError,
    Simulator,
    exported_symbols,
    load_library,
    sim_create,
    sim_destroy,
    sim_error_string,
    sim_generate,
    sim_generate_host,
    sim_update_scene,
    sim_replica,
    sim_debug_facets,
    sim_debug_echoes,
    sim_echoes_to_iq_static,
    sim_get_stats,
    sim_measure_pipe_peaks,
)
from .build import build_library  # noqa: F401
from .sharding import pulse_slab, gather_slabs  # noqa: F401
