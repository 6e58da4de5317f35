"""dpb_build_nlist_static (include/dpb.h): Alg. 1 with the kernels' scratch in a fixed file-scope
device array instead of the model's cudaMalloc'ed workspace, for callers that cannot allocate.  Checked against the
existing path (dpb_build_nlist) bit for bit — the formatted list is integer work — on two calls in a row that share the
scratch (the second on a DIFFERENT, smaller system, so stale contents of the first would show), and against the oracle.
The file sorts last on purpose (pytest -x: a failure here hides nothing behind it); it passes alone in a fresh process
and after the other tests."""
import numpy as np
import pytest

import gen
from gen.weights import MODELS

from conftest import small_model, random_box

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (the library has no CPU fallback)")
    return torch


def _both(m, coord, types, box):
    torch = _torch()
    dc = torch.tensor(coord, device="cuda")
    dt = torch.tensor(types.astype(np.int32), device="cuda")
    ref, ovf = m.build_nlist(dc, dt, box)
    out = torch.full((len(coord), m.nm), -7, dtype=torch.int32, device="cuda")
    status = torch.full((4,), -1, dtype=torch.int64, device="cuda")
    m.build_nlist_static(dc, dt, box, out, status)
    torch.cuda.synchronize()
    return ref.cpu().numpy(), ovf, out.cpu().numpy(), status.cpu().numpy()


def test_static_scratch_nlist_matches_the_allocating_path_twice_in_a_row():
    import paper_2004_11658_b200 as pk
    from oracle import Oracle
    torch = _torch()
    # call 1: BASELINE configs[0] (W192, 2 species, Nm = 138)
    spec = MODELS["W192"]
    coord, types, box = gen.make_system("W192")
    emb, fit = gen.make_weights(spec)
    m = pk.DPModel.from_spec(spec, emb, fit)
    ref, ovf, got, status = _both(m, coord, types, box)
    assert np.array_equal(got, ref), "call 1: the static-scratch list must equal dpb_build_nlist bit for bit"
    assert np.array_equal(got, Oracle.from_spec(spec, emb, fit).build_nlist(coord, types, box)[0])
    assert status[0] == (ref >= 0).sum() and status[1] == ovf == 0 and status[2] == 0 and status[3] > 0
    # call 2, right behind it on the same scratch: another model (3 species, short sections that overflow), fewer atoms
    spec2, emb2, fit2 = small_model(ntypes=3, s1=8, m_axis=4, fit_width=16, sel=(6, 9, 5), rcut=4.0, rcut_smth=1.0,
                                    seed=2, fit_scale=0.05)
    coord2, types2, box2 = random_box(90, 9.5, 3, seed=21, min_dist=1.1)
    m2 = pk.DPModel.from_spec(spec2, emb2, fit2)
    ref2, ovf2, got2, status2 = _both(m2, coord2, types2, box2)
    assert np.array_equal(got2, ref2), "call 2: stale scratch of call 1 must not leak"
    assert ovf2 > 0 and status2[1] == ovf2 and status2[0] == (ref2 >= 0).sum() and status2[2] == 0
    # call 3: the first system again (larger than call 2), and an empty input
    ref3, _, got3, status3 = _both(m, coord, types, box)
    assert np.array_equal(got3, ref) and np.array_equal(ref3, ref) and np.array_equal(status3, status)
    m.build_nlist_static(torch.empty((0, 3), dtype=torch.float64, device="cuda"),
                         torch.empty((0,), dtype=torch.int32, device="cuda"), box,
                         torch.empty((1, m.nm), dtype=torch.int32, device="cuda"))
    torch.cuda.synchronize()


def test_static_scratch_limits_and_deferred_errors():
    import paper_2004_11658_b200 as pk
    torch = _torch()
    spec = MODELS["W192"]
    emb, fit = gen.make_weights(spec)
    m = pk.DPModel.from_spec(spec, emb, fit)
    # beyond the stated maximum: a clear error, nothing launched, no allocation needed to find out
    n = 4097
    big = torch.zeros((n, 3), dtype=torch.float64, device="cuda")
    bt = torch.zeros((n,), dtype=torch.int32, device="cuda")
    out = torch.empty((n, m.nm), dtype=torch.int32, device="cuda")
    with pytest.raises(pk.DPBError, match="at most 4096 atoms"):
        m.build_nlist_static(big, bt, np.diag([40.0, 40.0, 40.0]).reshape(-1), out)
    n = 2000                                                   # 2000 * 138 slots > 262144
    with pytest.raises(pk.DPBError, match="at most 262144 slots"):
        m.build_nlist_static(big[:n].contiguous(), bt[:n].contiguous(), np.diag([40.0, 40.0, 40.0]).reshape(-1), out)
    with pytest.raises(pk.DPBError, match="exceeds the static scratch"):      # 30 x 30 x 30 cells x 2 types
        m.build_nlist_static(big[:8].contiguous(), bt[:8].contiguous(), np.diag([185.0, 185.0, 185.0]).reshape(-1), out)
    # a type index out of range is reported in status (the call never synchronises)
    coord, types, box = gen.make_system("W192")
    bad = types.astype(np.int32).copy()
    bad[5] = 2
    status = torch.zeros((4,), dtype=torch.int64, device="cuda")
    m.build_nlist_static(torch.tensor(coord, device="cuda"), torch.tensor(bad, device="cuda"), box,
                         torch.empty((len(coord), m.nm), dtype=torch.int32, device="cuda"), status)
    torch.cuda.synchronize()
    assert int(status[2].item()) & 1
