"""paper_2402_17248_b200 -- thin Python binding of libhb.so (include/hb.h).

B200-native (sm_100a) hybrid conventional/surrogate beamline push after Sandberg et al., PASC'24
(arXiv 2402.17248).  Every step of the path runs in the CUDA kernels of csrc/; this package only
marshals arguments: device pointers and the stream come from PyTorch tensors (torch is used for
device memory and streams, nothing else).  There is no CPU fallback: importing works anywhere, but
any call that needs the library fails loudly if libhb.so or a CUDA device is missing.
"""
from ._binding import (  # noqa: F401
    HbError, Lattice, lib, lib_path, moments, moments_static, to_device, to_host, allgather_merge_records,
    hb_lattice_create, hb_lattice_add_element, hb_lattice_set_element, hb_lattice_add_multipole, hb_lattice_add_surrogate, hb_lattice_set_run_mode,
    hb_lattice_set_centroid,
    hb_lattice_finalize, hb_lattice_num_monitors, hb_lattice_num_launches, hb_lattice_ref_bg_out,
    hb_push, hb_push_moments, hb_push_host, hb_push_candidates, hb_moments, hb_moments_scratch_bytes, hb_moments_merge, hb_lattice_destroy,
    hb_moments_static, hb_moments_static_max_particles,
    hb_lattice_enable_timing, hb_lattice_get_timing,
    hb_status_string, hb_last_error, hb_version, hb_surrogate_kernel, hb_device_peaks,
    ELEM_KINDS, ACTS, PRECS, COORDS, RUN_MODES, EXPORTED_SYMBOLS,
)
