"""Host logic of the seeded input generators (no method arithmetic lives there)."""
import torch

from paper_2603_14806_b200 import synth


def test_configs_follow_baseline_json():
    assert [c.N for c in synth.CONFIGS] == [64, 512, 2048, 4096, 8192]
    assert synth.CONFIGS[0].dtype == "f32" and all(c.dtype == "bf16" for c in synth.CONFIGS[1:])


def test_masks():
    m = synth.make_token_mask("tail", 512, 1001)
    assert m.sum().item() == 512 - 51 and m[-1] == 0 and m[0] == 1
    m = synth.make_token_mask("chains", 2048, 1002)
    assert m.sum().item() == 1900 and m[1899] == 1 and m[1900] == 0
    L = synth.chain_lengths(2048, 1002)
    assert len(L) == 4 and sum(L) == 1900 and min(L) >= 50
    m = synth.make_token_mask("scatter", 8192, 1004)
    assert m.sum().item() == 8192 - 410
    assert torch.equal(m, synth.make_token_mask("scatter", 8192, 1004))
    M = synth.pair_mask(synth.make_token_mask("tail", 64, 1), "bf16")
    assert M.dtype == torch.bfloat16 and M.shape == (64, 64) and M[0, 63] == 0 and M[0, 0] == 1


def test_params_and_z_seeded():
    p = synth.make_params(5, dtype="bf16")
    q = synth.make_params(5, dtype="bf16")
    assert all(torch.equal(p[k], q[k]) for k in p)
    assert p["w_a"].dtype == torch.bfloat16 and p["w_a"].shape == (128, 128)
    assert p["b_a"].dtype == torch.float32
    assert abs(p["w_a"].float().std().item() - 128 ** -0.5) < 0.01      # variance 1/fan_in (A5)
    assert abs(p["b_o"].std().item() - 0.02) < 0.01
    assert p["w_o"].float().abs().max() > 0                              # not zero-init
    r = synth.make_params(6, dtype="bf16")
    assert not torch.equal(p["w_a"], r["w_a"])
    z1 = synth.make_z(3, 16, 128, "bf16", chunk_rows=16)
    z2 = synth.make_z(3, 16, 128, "bf16", chunk_rows=16)
    assert torch.equal(z1, z2) and z1.shape == (16, 16, 128)
    assert abs(z1.float().std().item() - 1.0) < 0.05
    zf, Mf, pf = synth.make_inputs(synth.CONFIGS[0], 0)
    assert zf.dtype == torch.float32 and Mf.dtype == torch.float32 and pf["w_a"].dtype == torch.float32
