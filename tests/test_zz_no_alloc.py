"""GPU test of emu_bin_grains_noalloc (include/emu.h): binning for callers that cannot allocate device memory.

Some users of the library reach the point where a view must be binned without any way to obtain a workspace: the loop
that follows the microscope may not call cudaMalloc (it would wait for every stream of the GPU and hold up the camera
copies), a plug-in living beside a memory pool that already owns the whole GPU gets an out-of-memory error, and a
callee that is handed input and output tensors has no allocator to turn to.  For them the library carries a fixed 8 MiB
scratch block of its own.  This file checks that the entry point built on that block returns exactly what
emu_bin_grains returns with a caller's workspace - on two (in fact three) calls in a row, because the block is shared by
all calls and still holds what the previous call left behind - and that a batch beyond the limit is turned away with a
message that names the limit.

The file name sorts last on purpose: pytest -x stops at the first failure, so a failure here hides no other test.
"""
import numpy as np
import pytest

from emu_synth import CONFIGS, default_params, make_batch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def E():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    import paper_1311_5334_b200 as E
    E.exported_symbols()
    return E


def _case(cfg, n_views, cell_um, messy):
    b = make_batch(CONFIGS[cfg], cfg, n_views=n_views)
    p = default_params(cfg, cell_um=cell_um)
    g = b.grains.copy()
    if messy:                                       # grains outside the box are legal input (boundary cells), junk payloads too
        g[::7, 0] -= p["view_size_q"][0] // 3; g[::11, 1] += p["view_size_q"][1] // 2; g[::13, 2] -= 4000
        g[:, 3] = np.arange(len(g))[::-1] * 7 + 3
    return p, np.ascontiguousarray(g), b.view_off, b.n_views


def _bin_both_ways(E, p, g, view_off, n_views):
    """(sorted, cell_start, status) from the workspace path and from the no-allocation path, same inputs"""
    import torch
    prm = E.make_params(**{k: p[k] for k in ("view_size_q", "cell_size_q", "sep_min_q", "sep_max_q", "tube_r2_q", "min_grains")})
    d_g, d_off = torch.from_numpy(g).cuda(), torch.from_numpy(view_off).cuda()
    n_cells, _ = E.emu_grid_cells(prm)
    out = []
    for noalloc in (False, True):
        srt = torch.full((len(g), 4), -7, dtype=torch.int32, device="cuda")
        cs = torch.full((n_views * n_cells + 1,), -7, dtype=torch.int32, device="cuda")
        status = torch.zeros(1, dtype=torch.int64, device="cuda")
        if noalloc:
            E.emu_bin_grains_noalloc(prm, d_g, d_off, len(g), n_views, srt, cs, status)
        else:
            bin_bytes, _ = E.emu_workspace_bytes(prm, len(g), n_views)
            assert bin_bytes <= E.emu_bin_noalloc_max_bytes(), "test case too large for the built-in scratch"
            ws = torch.empty(bin_bytes + 256, dtype=torch.uint8, device="cuda")
            E.emu_bin_grains(prm, d_g, d_off, len(g), n_views, srt, cs, status, ws)
        torch.cuda.synchronize()
        out.append((srt.cpu().numpy(), cs.cpu().numpy(), int(status.cpu()[0])))
    return out


def test_noalloc_binning_equals_workspace_binning_on_calls_in_a_row(E, oracle_mod):
    # three calls that share the library's scratch block, each finding the leftovers of the one before:
    #  1. three config-4 views (193 k grains) in the bench's 3 x 4 x 4 um cells (114 k cells per view; the two-pass
    #     split + chunk kernels): 5.7 of the 8 MiB,
    #  2. three small config-0 views in coarse, skew cells with out-of-box grains (the one-block-per-view kernel) -
    #     a far smaller footprint, so most of the block still holds call 1's counters and staged grains,
    #  3. one config-1 view in the fine cells again.
    cases = [_case(4, 3, (3.0, 4.0, 4.0), False), _case(0, 3, (3.0, 17.0, 5.5), True), _case(1, 1, (3.0, 4.0, 4.0), True)]
    for p, g, view_off, n_views in cases:
        (s_ws, c_ws, st_ws), (s_na, c_na, st_na) = _bin_both_ways(E, p, g, view_off, n_views)
        assert st_ws == 0 and st_na == 0
        # integer work: the bar is bit-exact, as in test_binning_bit_exact
        assert np.array_equal(c_na, c_ws)
        assert np.array_equal(s_na, s_ws)
        # and both are the oracle's answer, so the comparison above is not two wrong results agreeing
        srt, cs = oracle_mod.bin_grains(p, g, view_off)
        assert np.array_equal(c_na, cs) and np.array_equal(s_na, srt)


def test_noalloc_binning_refuses_batches_beyond_its_scratch(E):
    import torch
    p = default_params(1, cell_um=(3.0, 4.0, 4.0))
    prm = E.make_params(**{k: p[k] for k in ("view_size_q", "cell_size_q", "sep_min_q", "sep_max_q", "tube_r2_q", "min_grains")})
    n_views, n = 64, 1 << 20
    bin_bytes, _ = E.emu_workspace_bytes(prm, n, n_views)
    assert bin_bytes > E.emu_bin_noalloc_max_bytes()
    n_cells, _ = E.emu_grid_cells(prm)
    d_g = torch.zeros((n, 4), dtype=torch.int32, device="cuda")
    d_off = torch.linspace(0, n, n_views + 1, device="cuda").to(torch.int32)
    srt = torch.full((n, 4), -7, dtype=torch.int32, device="cuda")
    cs = torch.full((n_views * n_cells + 1,), -7, dtype=torch.int32, device="cuda")
    status = torch.zeros(1, dtype=torch.int64, device="cuda")
    with pytest.raises(E.EmuError, match=r"EMU_ERR_CAPACITY") as err:
        E.emu_bin_grains_noalloc(prm, d_g, d_off, n, n_views, srt, cs, status)
    assert str(E.emu_bin_noalloc_max_bytes()) in str(err.value)
    torch.cuda.synchronize()
    assert int(srt.min()) == -7 and int(cs.min()) == -7 and int(status[0]) == 0      # nothing was enqueued
