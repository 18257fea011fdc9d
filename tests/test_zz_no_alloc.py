"""-m gpu: heom_level_max_static, the growth monitor with its scratch in a static __device__ array (no allocation,
depth <= HEOM_STATIC_MAX_DEPTH), against the existing heom_level_max path, on calls in a row that share the scratch.
Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu


def _levels_and_state(g):
    st = g.get_full_state()                                   # pinned order, [nodes][N][N] complex128
    lev = g.tables()[0].sum(axis=1).astype(np.uint8)          # level of every node, same order
    return st, lev


def _call(st_dev, lev_dev, out_dev, nodes, per, depth, stream):
    import torch
    from paper_1803_03498_b200 import level_max_static
    out_dev.fill_(float("nan"))                               # the kernel must write every entry
    torch.cuda.synchronize()
    level_max_static(st_dev.data_ptr(), lev_dev.data_ptr(), nodes, per, depth, out_dev.data_ptr(),
                     device=0, cuda_stream=stream.cuda_stream)
    stream.synchronize()
    return out_dev.cpu().numpy()


@pytest.mark.parametrize("name,D,steps", [("fmo", 4, 30), ("cfg5", 1, 3)])
def test_static_level_max_matches_existing_path_on_consecutive_calls(name, D, steps):
    import torch
    from paper_1803_03498_b200 import Heom
    w = (workloads.fmo_like() if name == "fmo" else workloads.get("cfg5")).with_(D=D)
    g = Heom(w.H_cm, w.lambda_cm, w.nu_per_fs, w.T_kelvin, w.K, w.D).bind()
    g.set_state(w.sigma0())
    g.rk4_steps(w.dt_fs, steps)
    per = g.N * g.N
    stream = torch.cuda.Stream()
    out = torch.empty(D + 1, dtype=torch.float64, device="cuda")

    # call 1: the state after `steps` steps
    want1 = g.level_max()
    st1, lev = _levels_and_state(g)
    lev_dev = torch.from_numpy(lev).cuda()
    st_dev = torch.from_numpy(st1.view(np.float64)).cuda()
    got1 = _call(st_dev, lev_dev, out, g.nodes, per, D, stream)
    assert np.array_equal(got1, want1)

    # call 2, straight after: a later state of the same propagation
    g.rk4_steps(w.dt_fs, steps)
    want2 = g.level_max()
    st2, _ = _levels_and_state(g)
    st_dev.copy_(torch.from_numpy(st2.view(np.float64)))
    free_before = torch.cuda.mem_get_info()[0]
    got2 = _call(st_dev, lev_dev, out, g.nodes, per, D, stream)
    assert np.array_equal(got2, want2)
    assert not np.array_equal(want1, want2)

    # call 3: every element 4x smaller than what the scratch last held -- stale maxima would survive a missing clear
    st_dev.mul_(0.25)
    got3 = _call(st_dev, lev_dev, out, g.nodes, per, D, stream)
    assert np.array_equal(got3, 0.25 * want2)
    assert torch.cuda.mem_get_info()[0] >= free_before        # nothing was allocated on the device

    # a NaN anywhere in a level reads as +inf, as on the existing path
    st_dev.view(-1)[2 * per * (g.nodes - 1) + 1] = float("nan")
    got4 = _call(st_dev, lev_dev, out, g.nodes, per, D, stream)
    assert np.isinf(got4[lev[-1]]) and np.array_equal(np.delete(got4, lev[-1]), np.delete(got3, lev[-1]))
    g.close()


def test_static_level_max_rejects_what_the_scratch_cannot_hold():
    import torch
    from paper_1803_03498_b200 import HeomError, STATIC_MAX_DEPTH, level_max_static
    st = torch.zeros(2 * 4 * 3, dtype=torch.float64, device="cuda")
    lev = torch.zeros(3, dtype=torch.uint8, device="cuda")
    out = torch.zeros(STATIC_MAX_DEPTH + 2, dtype=torch.float64, device="cuda")
    with pytest.raises(HeomError, match="depth 64 is outside 0..63"):
        level_max_static(st.data_ptr(), lev.data_ptr(), 3, 4, STATIC_MAX_DEPTH + 1, out.data_ptr())
    with pytest.raises(HeomError, match="NULL"):
        level_max_static(0, lev.data_ptr(), 3, 4, 2, out.data_ptr())
    with pytest.raises(HeomError, match="out of range"):
        level_max_static(st.data_ptr(), lev.data_ptr(), 3, 0, 2, out.data_ptr())
    # the largest depth it takes, an empty hierarchy level everywhere but L = 0
    level_max_static(st.data_ptr(), lev.data_ptr(), 3, 4, STATIC_MAX_DEPTH, out.data_ptr())
    torch.cuda.synchronize()
    assert float(out.abs().sum()) == 0.0
