"""tests/golden/c1_oracle_samples.txt: oracle-written regression values (see tests/golden/make_golden.py).
CPU: the oracle still reproduces them.  GPU: the CUDA path matches them within the parity tolerances."""
import importlib.util
import os

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
mg = importlib.util.module_from_spec(spec)
spec.loader.exec_module(mg)


def load():
    rows = np.loadtxt(os.path.join(HERE, "golden", "c1_oracle_samples.txt"))
    return rows[:, 0].astype(int), rows[:, 1:4], rows[:, 4:7], rows[:, 7:10]


def test_oracle_reproduces_golden():
    ids, f0, x5, v5 = load()
    assert list(ids) == mg.IDS
    g0, gx, gv = mg.compute()
    assert np.abs(g0 - f0).max() < 1e-9 and np.abs(gx - x5).max() < 1e-10 and np.abs(gv - v5).max() < 1e-9


@pytest.mark.gpu
def test_gpu_matches_golden():
    torch = pytest.importorskip("torch")
    from paper_2302_02474_b200 import inputs, tild
    ids, f0, x5, v5 = load()
    cfg = inputs.C1
    st = inputs.make_state(cfg)
    eng = tild.Tild(tild.params_from_config(cfg))
    d = lambda a: torch.from_numpy(a).cuda()
    eng.tild_set_state(d(st.x), d(st.v), d(st.type), d(st.bond_partner), 0)
    _, _, f, _ = eng.tild_get_state(want_v=False, want_f=True)
    f = f.cpu().numpy()[ids]
    assert np.abs(f - f0).max() <= 1e-5 * 25.0          # RMS force of C1 is ~25; tolerance of DESIGN.md A19
    eng.tild_step(mg.NSTEPS)
    x, v, _, step = eng.tild_get_state()
    assert step == mg.NSTEPS
    dx = x.cpu().numpy()[ids].astype(np.float64) - x5
    dx -= 10.0 * np.round(dx / 10.0)
    assert np.abs(dx).max() <= 1e-4 and np.abs(v.cpu().numpy()[ids] - v5).max() <= 2e-3
