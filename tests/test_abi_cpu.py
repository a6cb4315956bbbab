"""CPU checks of the boundary: libemu4pi.so loads without a GPU, exports every function include/emu.h declares, and
its host-only entry points (no CUDA call inside) validate their arguments."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def E():
    from paper_1311_5334_b200 import build as lib_build
    lib_build.build()                        # nvcc cross-compiles sm_100a without a GPU
    import paper_1311_5334_b200 as E
    return E


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "emu.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"^\s*(?:size_t|int64_t|int|void|emu_profile\s*\*|emu_stream\s*\*)\s+\**\s*(emu_\w+)\s*\(", src, flags=re.M)
    return sorted(set(names))


def test_every_declared_symbol_is_exported(E):
    declared = _declared_functions()
    assert len(declared) >= 13 and "emu_bin_grains" in declared and "emu_find_tracks" in declared and "emu_fit_tracks" in declared
    lib = C.CDLL(E.library_path())
    for name in declared:
        getattr(lib, name)                   # AttributeError if the symbol is missing
    assert sorted(E.exported_symbols()) == declared, "binding and header disagree on the entry points"


def test_struct_sizes_match_the_header(E):
    from paper_1311_5334_b200.binding import emu_params
    assert C.sizeof(emu_params) == 4 * (1 + 3 + 3 + 6 + 4 + 8)
    assert E.TRACK_DTYPE.itemsize == 32 and E.FIT_DTYPE.itemsize == 48


def test_host_only_calls(E):
    # the paper's own geometry: 1280 x 1024 px x 40 frames in cells of 32 x 32 px x 1 frame = 51 200 cells
    prm = E.make_params((1280, 1024, 40), (32, 32, 1), 1, 25, 1, 5)
    n, dims = E.emu_grid_cells(prm)
    assert n == 51200 and dims == (40, 32, 40)
    prm = E.make_params((22400, 19200, 3200), (256, 256, 256), 256, 1280, 2621, 8)
    bin_b, find_b = E.emu_workspace_bytes(prm, 64000, 1)
    assert bin_b >= 64000 * 16 and find_b > 0
    assert E.emu_host_arena_bytes(prm, 64000, 1) > bin_b
    # documented range violations -> EMU_ERR_INVALID
    for bad in (dict(tube_ext_q=-2), dict(min_grains=1), dict(sep_max_q=4096)):
        kw = dict(view_size_q=(22400, 19200, 3200), cell_size_q=(256, 256, 256), sep_min_q=256, sep_max_q=1280,
                  tube_r2_q=2621, min_grains=8)
        kw.update(bad)
        with pytest.raises(E.EmuError):
            E.emu_workspace_bytes(E.make_params(**kw), 10, 1)


def test_compute_calls_refuse_host_tensors(E):
    import torch
    prm = E.make_params((6400, 6400, 3200), (256, 256, 256), 256, 1280, 2621, 8)
    t = torch.zeros((4, 4), dtype=torch.int32)
    with pytest.raises(E.EmuError):          # no CPU fallback: a host tensor is an error, not a slow path
        E.emu_bin_grains(prm, t, t, 4, 1, t, t, t, t)


def test_microbenchmark_compiles_for_sm100a(tmp_path):
    """microbench/mb_pipes.cu (the measured issue peak bench.py reports) is not part of build(); it must still compile"""
    from paper_1311_5334_b200 import build as lib_build
    exe = lib_build.build_microbench(str(tmp_path))
    assert os.path.exists(exe) and os.path.getsize(exe) > 0
