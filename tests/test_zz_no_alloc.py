"""tild_cell_start_noalloc (include/tild.h): the cell offsets of the a1 index map from a context-free entry point that
allocates nothing -- its scan partials live in a static __device__ array of the library.  Checked against the existing
path (tild_index_map with a context) and against the oracle's counting sort, bit for bit, on two calls in a row (the
calls share the static array).  Collected last on purpose: the run uses `pytest -x`."""
import numpy as np
import pytest

from oracle import tild_oracle as orc
from paper_2302_02474_b200 import inputs, tild
from tild_test_util import oracle_params, small_cfg

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def reference_offsets(cfg):
    """(cell_key, cell_start) of the existing path, as CUDA int32 tensors holding uint32, + the oracle's cell_start."""
    st = inputs.make_state(cfg)
    eng = tild.Tild(tild.params_from_config(cfg))
    _, key, _, start = eng.tild_index_map(torch.from_numpy(st.x).cuda())
    okey = orc.index_map(oracle_params(cfg), st.x)[2]
    _, ostart = orc.cell_sort(cfg.n, cfg.M, okey)
    key, start = key.clone(), start.clone()       # the engine's outputs outlive it
    eng.close()
    return key, start, ostart


def test_two_calls_in_a_row_match_the_context_path_bit_for_bit():
    # two different meshes, the second larger than one scan block (4096 entries) by a ragged amount and with empty cells
    cfgs = [small_cfg(order=2), small_cfg(order=3, grid=(40, 36, 50), box=(20.0, 18.0, 25.0), n_chains=700)]
    refs = [reference_offsets(c) for c in cfgs]
    assert cfgs[0].M + 1 > 4096 and (cfgs[1].M + 1) % 4096 != 0 and cfgs[1].M > 16 * 4096
    outs, bads = [], []
    for cfg, (key, _, _) in zip(cfgs, refs):      # back to back on one stream, no synchronisation in between
        out = torch.full((cfg.M + 1,), -1, dtype=torch.int32, device="cuda")
        bad = torch.full((1,), -1, dtype=torch.int32, device="cuda")
        tild.tild_cell_start_noalloc(key, cfg.M, out, bad)
        outs.append(out)
        bads.append(bad)
    torch.cuda.synchronize()
    for cfg, (key, start, ostart), out, bad in zip(cfgs, refs, outs, bads):
        assert torch.equal(out, start)
        assert np.array_equal(out.cpu().numpy().view(np.uint32), ostart)
        assert int(bad.item()) == 0
        assert int(out[-1].item()) == cfg.n
    # the same input again after the other one has used the array: nothing of the previous call is left in it
    again = torch.empty_like(outs[0])
    tild.tild_cell_start_noalloc(refs[0][0], cfgs[0].M, again)
    assert torch.equal(again, refs[0][1])


def test_keys_outside_the_mesh_are_left_out_and_counted():
    cfg = small_cfg(order=2)
    key, start, _ = reference_offsets(cfg)
    half = cfg.M // 2
    out = torch.empty((half + 1,), dtype=torch.int32, device="cuda")
    bad = torch.zeros((1,), dtype=torch.int32, device="cuda")
    tild.tild_cell_start_noalloc(key, half, out, bad)
    assert torch.equal(out, start[: half + 1])    # offsets of the cells that are inside are unchanged
    assert int(bad.item()) == cfg.n - int(start[half].item())


def test_empty_input_and_sizes_beyond_the_static_array():
    out = torch.full((17,), -1, dtype=torch.int32, device="cuda")
    tild.tild_cell_start_noalloc(torch.empty((0,), dtype=torch.int32, device="cuda"), 16, out)
    assert int(out.abs().sum().item()) == 0
    with pytest.raises(tild.TildError, match="TILD_NOALLOC_MAX_CELLS"):
        tild.tild_cell_start_noalloc(torch.zeros((4,), dtype=torch.int32, device="cuda"), tild.NOALLOC_MAX_CELLS + 1, out)
    assert int(out.abs().sum().item()) == 0       # rejected before anything was launched


def test_the_largest_supported_mesh():
    n_cells = tild.NOALLOC_MAX_CELLS              # a 256^3 mesh: 4097 scan blocks, all of the static array
    g = torch.Generator(device="cuda").manual_seed(7)
    key = torch.randint(0, n_cells, (1 << 20,), generator=g, device="cuda", dtype=torch.int32)
    out = torch.empty((n_cells + 1,), dtype=torch.int32, device="cuda")
    tild.tild_cell_start_noalloc(key, n_cells, out)
    counts = torch.bincount(key.long(), minlength=n_cells)
    ref = torch.zeros((n_cells + 1,), dtype=torch.int64, device="cuda")
    ref[1:] = torch.cumsum(counts, 0)
    assert torch.equal(out.long(), ref)
