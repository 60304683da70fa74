"""The whole-tensor parity harness (tests/parity_util.py) checked on the CPU: walking the tensor
block by block must give exactly the errors a direct whole-tensor comparison gives, and must find a
planted outlier.  No GPU needed; the arithmetic is the oracle's."""
import numpy as np
import pytest
import torch

import parity_util as U
from oracle import trimul_oracle as orc
from paper_2603_14806_b200 import synth


@pytest.mark.parametrize("direction", [orc.OUTGOING, orc.INCOMING])
def test_block_walk_equals_direct_comparison(direction, tmp_path, monkeypatch):
    monkeypatch.setenv("FOLDCP_PARITY_LOG", str(tmp_path / "rec.jsonl"))
    N = 40
    cfg = synth.CONFIGS[1]
    z, _, p = synth.make_inputs(cfg, direction, "cpu", N=N)
    M = synth.pair_mask(synth.make_token_mask("scatter", N, 3), "bf16")
    ref = U.oracle_full(z, M, p, direction)
    rng = np.random.default_rng(0)
    got = ref + 1e-3 * rng.standard_normal(ref.shape)
    got[17, 5, 99] += 0.5                                       # planted outlier
    e = U.whole_tensor_errors(torch.from_numpy(got), z, M, p, direction, block_rows=7)
    d = got - ref
    assert e["outputs"] == ref.size and e["finite"]
    assert abs(e["rel_fro"] - np.linalg.norm(d) / np.linalg.norm(ref)) < 1e-12
    assert abs(e["max_over_rms"] - np.abs(d).max() / np.sqrt(np.mean(ref ** 2))) < 1e-9
    assert e["argmax"] == [17, 5, 99]
    # a subset of row blocks: rms and errors over those rows only
    e2 = U.whole_tensor_errors(torch.from_numpy(got), z, M, p, direction, row_blocks=[(3, 9), (30, 40)])
    rows = np.r_[3:9, 30:40]
    assert e2["outputs"] == ref[rows].size
    assert abs(e2["rel_fro"] - np.linalg.norm(d[rows]) / np.linalg.norm(ref[rows])) < 1e-12
    # a sorted row subset through the compacted-a path (the N = 8192 form)
    sel = np.array([1, 4, 5, 17, 22, 39])
    e3 = U.whole_tensor_errors(torch.from_numpy(got), z, M, p, direction, rows=sel, block_rows=4)
    assert e3["outputs"] == ref[sel].size and e3["argmax"] == [17, 5, 99]
    assert abs(e3["rel_fro"] - np.linalg.norm(d[sel]) / np.linalg.norm(ref[sel])) < 1e-12
    assert abs(e3["max_over_rms"] - np.abs(d[sel]).max() / np.sqrt(np.mean(ref[sel] ** 2))) < 1e-9
    rec = U.record_parity("harness", e, "bf16", N=N)
    assert rec["margin_max_over_rms"] < 0 and (tmp_path / "rec.jsonl").read_text().count("\n") == 1
