"""Host logic of the brute-force plan tuner (SURVEY 8 f NEXT-4) and the plan-file round trip."""
import numpy as np
import pytest

from paper_1305_0036_b200 import tuner as T
from paper_1305_0036_b200 import workloads as W


def test_compositions_cover_exactly_the_valid_splits():
    for total in (1, 5, 9, 10, 18, 21):
        comps = list(T.compositions(total, 9, 4))
        assert len(set(comps)) == len(comps)
        assert all(sum(c) == total and 1 <= len(c) <= 4 and all(1 <= b <= 9 for b in c) for c in comps)
        brute = [c for k in range(1, 5) for c in np.ndindex(*([9] * k)) if sum(b + 1 for b in c) == total]
        assert len(comps) == len(brute)
    assert list(T.compositions(0)) == [()]
    assert list(T.compositions(40, 9, 4)) == []          # does not fit four groups of nine


def test_candidates_put_the_default_plan_first_and_stay_bounded():
    for N in (13, 22, 27, 30, 32, 33):
        c = T.candidates(N)
        assert 0 < len(c) <= 48
        assert all(sum(p["groups"]) == N - 12 for p in c)
        assert all(p["chunk"] == 0 or (len(p["groups"]) >= 2 and 12 + p["groups"][0] <= 21) for p in c)
    assert T.candidates(30)[0]["groups"] == [9, 9] and T.candidates(30)[0]["chunk"] == 1 and T.candidates(30)[0]["kernel"] == 1
    assert {p["kernel"] for p in T.candidates(30)} == {1}
    assert T.candidates(27)[0]["groups"] == [9, 6]


def test_plan_line_format():
    line = T.plan_line(30, {"groups": [9, 9], "chunk": 1, "l2_promotion": 2, "kernel": 1})
    assert line == "N=30 groups=9,9 kernel=1 chunk=1 chunk_max_log2=21 chunk_min_log2=21 l2_promotion=2"
    assert "chunk_min_log2=16" in T.plan_line(20, {"groups": [4, 2, 2], "chunk": 1, "l2_promotion": 0, "kernel": 1})


@pytest.mark.gpu
def test_plan_file_round_trip_through_the_c_abi(tmp_path):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from oracle import ts_oracle as O
    from paper_1305_0036_b200 import binding as B
    path = tmp_path / "test.plan"
    path.write_text("# comment\nN=18 groups=3,3 kernel=1 chunk=0 chunk_max_log2=21 l2_promotion=0\n"
                    + T.plan_line(20, {"groups": [4, 2, 2], "chunk": 1, "l2_promotion": 0, "kernel": 1}) + "\n")
    w = W.generic(20, seed=2020, tau=0.02, n_steps=2)
    ts = B.TrotterSuzuki(20, w.h, w.J)
    ts.load_plan_file(path)
    plan = ts.describe_plan()
    assert "H[spins 12..15" in plan and "H[spins 16..17" in plan and "H[spins 18..19" in plan and "L2-blocked" in plan
    ts.set_state(w.state())
    ts.evolve(w.tau, 2, 4)
    ref = w.state()
    O.evolve(ref, 20, w.h, w.J, w.tau, 2, 4, True)
    assert np.max(np.abs(ts.get_state() - ref)) <= 1e-11
    ts.close()
    ts = B.TrotterSuzuki(19, *[W.generic(19, seed=1).h, W.generic(19, seed=1).J])
    before = ts.describe_plan()
    ts.load_plan_file(path)                       # no line for N = 19: nothing changes
    assert ts.describe_plan() == before
    with pytest.raises(B.TSError):
        ts.load_plan_file(tmp_path / "missing.plan")
    ts.close()
