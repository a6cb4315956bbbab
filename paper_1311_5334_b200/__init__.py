"""paper_1311_5334_b200 - B200-native 4pi emulsion track finding (Ariga & Ariga, arXiv 1311.5334).

The product is the C-ABI library libemu4pi.so (include/emu.h; kernels in csrc/).  This package is
the thin Python binding: the same entry points by the same names, argument marshalling only.
PyTorch supplies device memory and streams, nothing else.  There is no CPU fallback: without the
built library, or without a CUDA device for the compute calls, everything here raises.
"""
from .binding import (EMU_CNT, EMU_ST, EMU_STAGE, HostPath, StreamPath, Profile, emu_host_arena_bytes, FIT_DTYPE, TRACK_DTYPE, EmuError, PathBuffers, PathResult, emu_bin_grains,
                      emu_count_seeds, emu_find_tracks, emu_fit_tracks, emu_grid_cells, emu_workspace_bytes,
                      emu_recognize_grains, emu_recognize_ws_bytes, emu_bin_grains_noalloc, emu_bin_noalloc_max_bytes,
                      exported_symbols, library_path, make_params, run_path)

__all__ = ["EMU_CNT", "EMU_ST", "EMU_STAGE", "HostPath", "StreamPath", "Profile", "emu_host_arena_bytes", "FIT_DTYPE", "TRACK_DTYPE", "EmuError", "PathBuffers", "PathResult",
           "emu_bin_grains", "emu_count_seeds", "emu_find_tracks", "emu_fit_tracks", "emu_grid_cells",
           "emu_workspace_bytes", "emu_bin_grains_noalloc", "emu_bin_noalloc_max_bytes", "emu_recognize_grains", "emu_recognize_ws_bytes", "exported_symbols", "library_path", "make_params", "run_path"]
