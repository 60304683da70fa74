"""GPU parity tests proper: the CUDA path (through the C ABI) against the fp64 oracle, element by
element on the same seeded inputs.  Small sizes use the full oracle; BASELINE.json's large configs
use the sub-grid oracle (exact full-k sums on sampled rows x columns)."""
import numpy as np
import pytest
import torch

import parity_util as U
from paper_2603_14806_b200 import binding as B
from paper_2603_14806_b200 import synth

pytestmark = pytest.mark.gpu
DEV = "cuda"
OUT, INC = B.OUTGOING, B.INCOMING


def to_dev(p):
    return {k: v.to(DEV) for k, v in p.items()}


def run_full(cfg, direction, N=None, mask_output=True, mask_kind=None):
    z, M, p = synth.make_inputs(cfg, direction, "cpu", N=N)
    if mask_kind is not None:
        M = synth.pair_mask(synth.make_token_mask(mask_kind, z.shape[0], cfg.seed), cfg.dtype)
    ref = U.oracle_full(z, M, p, direction, mask_output=mask_output)
    out = B.trimul(z.to(DEV), M.to(DEV), to_dev(p), direction, mask_output=mask_output)
    torch.cuda.synchronize()
    return U.assert_parity(U.np64(out), ref, cfg.dtype, f"cfg{cfg.index} N={z.shape[0]} dir={direction}")


# ---------------------------------------------------------------- BASELINE configs 0 and 1 (full oracle)
@pytest.mark.parametrize("direction", [OUT, INC])
def test_config0_fp32_n64(direction):
    e = run_full(synth.CONFIGS[0], direction)
    assert e["rel_fro"] < 1e-5


@pytest.mark.parametrize("direction", [OUT, INC])
@pytest.mark.parametrize("mask_output", [True, False])
def test_config1_bf16_n512(direction, mask_output):
    run_full(synth.CONFIGS[1], direction, mask_output=mask_output)


# ---------------------------------------------------------------- ragged / tiny / odd sizes (full oracle)
@pytest.mark.parametrize("N", [8, 72, 136, 328])
@pytest.mark.parametrize("direction", [OUT, INC])
def test_bf16_ragged_sizes(N, direction):
    # 328 = 2 full 128-tiles + a 72 tail, not a multiple of the 64-wide k block either
    run_full(synth.CONFIGS[1], direction, N=N, mask_kind="scatter")


@pytest.mark.parametrize("N", [1, 5, 12, 67])
@pytest.mark.parametrize("direction", [OUT, INC])
def test_fp32_odd_sizes(N, direction):
    run_full(synth.CONFIGS[0], direction, N=N, mask_kind="tail" if N >= 10 else "ones")


# ---------------------------------------------------------------- stage-level parity
@pytest.mark.parametrize("direction", [OUT, INC])
@pytest.mark.parametrize("N", [64, 328, 520])
@pytest.mark.parametrize("ab_dtype", [torch.bfloat16, torch.float16])
def test_contract_stage_bf16(direction, N, ab_dtype):
    """a, b as bf16 (the gradient GEMMs' format) and as fp16 (what the project stage writes on the
    forward path); o is bf16 in both cases."""
    from oracle import trimul_oracle as orc
    g = torch.Generator().manual_seed(N + direction)
    a = torch.randn(128, N, N, generator=g).to(ab_dtype)
    b = torch.randn(128, N, N, generator=g).to(ab_dtype)
    o = B.contract(a.to(DEV), b.to(DEV), direction)
    torch.cuda.synchronize()
    assert o.dtype == torch.bfloat16
    ref = orc.contraction(np.transpose(U.np64(a), (1, 2, 0)), np.transpose(U.np64(b), (1, 2, 0)), direction)
    got = np.transpose(U.np64(o), (1, 2, 0))
    # only the final bf16 rounding of o (2^-9 relative) plus fp32 accumulation
    assert np.abs(got - ref).max() <= 2.0 ** -8 * np.abs(ref).max()
    assert U.errors(got, ref)["rel_fro"] < 3e-3


def test_project_stage_bf16():
    from oracle import trimul_oracle as orc
    cfg = synth.CONFIGS[1]
    z, M, p = synth.make_inputs(cfg, OUT, "cpu", N=136)
    a, b = B.project(z.to(DEV), M.to(DEV), to_dev(p))
    torch.cuda.synchronize()
    assert a.dtype == torch.float16 and b.dtype == torch.float16     # fp16 intermediates in bf16 mode
    q = U.params64(p)
    zp = orc.layer_norm(U.np64(z), q["ln_in_gamma"], q["ln_in_beta"], 1e-5)
    ra = orc.gated_projection(zp, U.np64(M), q["w_a"], q["b_a"], q["w_a_gate"], q["b_a_gate"])
    rb = orc.gated_projection(zp, U.np64(M), q["w_b"], q["b_b"], q["w_b_gate"], q["b_b_gate"])
    for got, ref in ((a, ra), (b, rb)):
        e = U.errors(np.transpose(U.np64(got), (1, 2, 0)), ref)
        # fp16 storage (2^-12 relative) + fp16 operand tiles + tanh.approx gates
        assert e["rel_fro"] < 2e-3 and e["max_over_rms"] < 2e-2, e


@pytest.mark.parametrize("mask_output", [True, False])
def test_finalize_stage_bf16(mask_output):
    """K3 alone: random channel-major o (with per-channel offsets, so LN(o) has work to do)."""
    from oracle import trimul_oracle as orc
    cfg = synth.CONFIGS[1]
    N = 136
    z, M, p = synth.make_inputs(cfg, OUT, "cpu", N=N)
    M = synth.pair_mask(synth.make_token_mask("scatter", N, cfg.seed), cfg.dtype)
    g = torch.Generator().manual_seed(7)
    o = (torch.randn(128, N, N, generator=g) * 3 + torch.randn(128, 1, 1, generator=g)).to(torch.bfloat16)
    out = B.finalize(o.to(DEV), z.to(DEV), M.to(DEV), to_dev(p), mask_output=mask_output)
    torch.cuda.synchronize()
    q = U.params64(p)
    zp = orc.layer_norm(U.np64(z), q["ln_in_gamma"], q["ln_in_beta"], 1e-5)
    ref = orc.output_stage(np.transpose(U.np64(o), (1, 2, 0)), zp, U.np64(M), q, 1e-5, mask_output)
    e = U.errors(U.np64(out), ref)
    # only the output rounding (2^-9 relative) plus fp16 operand tiles and fp32 accumulation
    assert e["rel_fro"] < 3e-3 and e["max_over_rms"] < 5e-2


# ---------------------------------------------------------------- the stages in the form the fused call chains them
def test_project_stats_stage():
    """foldcp_trimul_project_stats: a, b bitwise those of foldcp_trimul_project, plus (mean, rstd) of
    LayerNorm(z) per pair against the fp64 definition."""
    cfg = synth.CONFIGS[1]
    N = 136
    z, M, p = synth.make_inputs(cfg, OUT, "cpu", N=N)
    a0, b0 = B.project(z.to(DEV), M.to(DEV), to_dev(p))
    a1, b1, st = B.project_stats(z.to(DEV), M.to(DEV), to_dev(p))
    torch.cuda.synchronize()
    assert torch.equal(a0, a1) and torch.equal(b0, b1)
    zz = U.np64(z)
    mean = zz.mean(axis=-1)
    rstd = 1.0 / np.sqrt(zz.var(axis=-1) + 1e-5)          # biased variance, eps inside the sqrt (A6)
    got = U.np64(st)
    assert np.abs(got[..., 0] - mean).max() <= 1e-6 * max(1.0, np.abs(mean).max())
    assert np.abs(got[..., 1] / rstd - 1.0).max() <= 1e-5


@pytest.mark.parametrize("direction", [OUT, INC])
@pytest.mark.parametrize("N", [64, 328])
def test_contract_stage_fused_o(direction, N):
    """FOLDCP_BF16_F16ALL: o leaves K2 as fp16, multiplied by foldcp_trimul_o_scale(N) (a power of two
    ~ 1/sqrt(N)): only fp16's 2^-11 rounding separates it from the fp64 contraction."""
    from oracle import trimul_oracle as orc
    g = torch.Generator().manual_seed(N + direction)
    a = torch.randn(128, N, N, generator=g).to(torch.float16)
    b = torch.randn(128, N, N, generator=g).to(torch.float16)
    o = B.contract(a.to(DEV), b.to(DEV), direction, fused_o=True)
    torch.cuda.synchronize()
    assert o.dtype == torch.float16
    sc = B.o_scale(N)
    assert sc == 2.0 ** -int(np.ceil(np.log2(N) / 2))
    ref = sc * orc.contraction(np.transpose(U.np64(a), (1, 2, 0)), np.transpose(U.np64(b), (1, 2, 0)), direction)
    got = np.transpose(U.np64(o), (1, 2, 0))
    assert np.abs(got - ref).max() <= 2.0 ** -10 * np.abs(ref).max()
    assert U.errors(got, ref)["rel_fro"] < 5e-4


@pytest.mark.parametrize("mask_output", [True, False])
@pytest.mark.parametrize("with_stats", [True, False])
def test_finalize_fused_stage(mask_output, with_stats):
    """K3 as the fused call launches it: o in fp16 scaled by o_scale(N) (LayerNorm(o) must absorb the
    scale through eps), LayerNorm(z) statistics handed over by K1 or recomputed."""
    from oracle import trimul_oracle as orc
    cfg = synth.CONFIGS[1]
    N = 136
    z, M, p = synth.make_inputs(cfg, OUT, "cpu", N=N)
    M = synth.pair_mask(synth.make_token_mask("scatter", N, cfg.seed), cfg.dtype)
    g = torch.Generator().manual_seed(7)
    o64 = (torch.randn(128, N, N, generator=g) * 3 + torch.randn(128, 1, 1, generator=g)).double()
    sc = B.o_scale(N)
    o16 = (o64 * sc).to(torch.float16)
    stats = None
    if with_stats:
        _, _, stats = B.project_stats(z.to(DEV), M.to(DEV), to_dev(p))
    out = B.finalize_fused(o16.to(DEV), z.to(DEV), stats, M.to(DEV), to_dev(p), mask_output=mask_output)
    torch.cuda.synchronize()
    q = U.params64(p)
    zp = orc.layer_norm(U.np64(z), q["ln_in_gamma"], q["ln_in_beta"], 1e-5)
    # the oracle sees the values the kernel was given, unscaled: o16 / sc is exact (power of two)
    ref = orc.output_stage(np.transpose(o16.double().numpy() / sc, (1, 2, 0)), zp, U.np64(M), q, 1e-5, mask_output)
    e = U.errors(U.np64(out), ref)
    U.record_parity(f"finalize_fused stage N={N} mask_output={mask_output} stats={'K1' if with_stats else 'recomputed'}",
                    e, "bf16", N=N)
    assert e["rel_fro"] < 3e-3 and e["max_over_rms"] < 5e-2


@pytest.mark.parametrize("direction", [OUT, INC])
def test_fused_stage_chain_is_the_full_call_bitwise(direction):
    """project_stats -> contract (fp16 scaled o) -> finalize_fused are exactly the three launches of
    foldcp_trimul in bf16 mode."""
    cfg = synth.CONFIGS[1]
    N = 264
    z, M, p = synth.make_inputs(cfg, direction, "cpu", N=N)
    zd, Md, pd = z.to(DEV), M.to(DEV), to_dev(p)
    a, b, st = B.project_stats(zd, Md, pd)
    o = B.contract(a, b, direction, fused_o=True)
    out = B.finalize_fused(o, zd, st, Md, pd)
    full = B.trimul(zd, Md, pd, direction)
    torch.cuda.synchronize()
    assert torch.equal(out, full)


@pytest.mark.parametrize("direction", [OUT, INC])
def test_bf16_n1024_full_tensor(direction):
    """Whole-tensor parity at N = 1024 (1.3e8 outputs): the max-abs criterion is the binding one
    and grows with the number of outputs (SURVEY 8(c) error budget), so it is checked on a full
    tensor, not only on sub-grids."""
    e = run_full(synth.CONFIGS[1], direction, N=1024, mask_kind="tail")
    assert e["rel_fro"] < 5e-3


# ---------------------------------------------------------------- NEXT-1: residual-fused and batched forms
@pytest.mark.parametrize("cfg_i,N", [(0, 67), (1, 264)])
@pytest.mark.parametrize("direction", [OUT, INC])
def test_residual_fused(cfg_i, N, direction):
    """out = z + update (PAPER.md lines 121-128 write the update as `z_nm +=`), fused into K3."""
    from oracle import trimul_oracle as orc
    cfg = synth.CONFIGS[cfg_i]
    z, M, p = synth.make_inputs(cfg, direction, "cpu", N=N)
    M = synth.pair_mask(synth.make_token_mask("tail", N, cfg.seed), cfg.dtype)
    ref_u = U.oracle_full(z, M, p, direction)
    ref = orc.trimul_residual(U.np64(z), U.np64(M), U.params64(p), direction)
    out = B.trimul(z.to(DEV), M.to(DEV), to_dev(p), direction, residual=True)
    torch.cuda.synchronize()
    got = U.np64(out)
    assert np.all(np.isfinite(got))
    # the error budget is the update's (north_star tolerance on the update) plus the rounding of
    # the sum to the output dtype (half an ulp of |z + update|)
    ulp = 2.0 ** -8 if cfg.dtype == "bf16" else 2.0 ** -23
    rms_u = np.sqrt(np.mean(ref_u ** 2))
    tol = U.TOL[cfg.dtype]["max_over_rms"] * rms_u + 0.5 * ulp * np.abs(ref).max()
    assert np.abs(got - ref).max() <= tol
    assert np.linalg.norm(got - ref) / np.linalg.norm(ref) <= U.TOL[cfg.dtype]["rel_fro"]


@pytest.mark.parametrize("residual", [False, True])
def test_batched_equals_single_calls_bitwise(residual):
    cfg = synth.CONFIGS[1]
    N, Bn = 136, 3
    zs, Ms = [], []
    for b in range(Bn):
        z, _, p = synth.make_inputs(cfg, OUT, "cpu", N=N)
        g = torch.Generator().manual_seed(100 + b)
        zs.append((z.float() + 0.25 * torch.randn(z.shape, generator=g)).to(z.dtype))
        Ms.append(synth.pair_mask(synth.make_token_mask("scatter", N, cfg.seed + b), cfg.dtype))
    zb, Mb, pd = torch.stack(zs).to(DEV), torch.stack(Ms).to(DEV), to_dev(p)
    out_b = B.trimul(zb, Mb, pd, INC, residual=residual)
    singles = [B.trimul(zb[b].contiguous(), Mb[b].contiguous(), pd, INC, residual=residual)
               for b in range(Bn)]
    torch.cuda.synchronize()
    assert out_b.shape == zb.shape
    for b in range(Bn):
        assert torch.equal(out_b[b], singles[b])
    e = U.errors(U.np64(out_b[1]) - (U.np64(zb[1]) if residual else 0.0),
                 U.oracle_full(zs[1], Ms[1], p, INC))
    assert e["rel_fro"] < 1e-2 + (2e-2 if residual else 0.0)


# ---------------------------------------------------------------- NEXT-2 (part): contraction backward
@pytest.mark.parametrize("direction", [OUT, INC])
@pytest.mark.parametrize("N,dtype", [(64, torch.bfloat16), (328, torch.bfloat16), (520, torch.bfloat16),
                                     (67, torch.float32)])
def test_contract_backward_stage(direction, N, dtype):
    from oracle import trimul_oracle as orc
    g = torch.Generator().manual_seed(3 * N + direction)
    a, b, d_o = (torch.randn(128, N, N, generator=g).to(dtype) for _ in range(3))
    d_a, d_b = B.contract_backward(d_o.to(DEV), a.to(DEV), b.to(DEV), direction)
    torch.cuda.synchronize()
    t = lambda x: np.transpose(U.np64(x), (1, 2, 0))
    ra, rb = orc.contraction_backward(t(d_o), t(a), t(b), direction)
    for got, ref in ((t(d_a), ra), (t(d_b), rb)):
        if dtype == torch.bfloat16:
            # only the final bf16 rounding (2^-9 relative) plus fp32 accumulation
            assert np.abs(got - ref).max() <= 2.0 ** -8 * np.abs(ref).max()
            assert U.errors(got, ref)["rel_fro"] < 3e-3
        else:
            assert U.errors(got, ref)["rel_fro"] < 1e-5


# ---------------------------------------------------------------- BASELINE configs 2-4 (sub-grid oracle)
def run_subgrid(cfg, direction, n_idx, seed):
    N = cfg.N
    z = synth.make_z(cfg.seed, N, cfg.c_z, cfg.dtype, DEV)
    m = synth.make_token_mask(cfg.mask_kind, N, cfg.seed)
    M = synth.pair_mask(m, cfg.dtype, DEV)
    p = to_dev(synth.make_params(cfg.seed * 2 + direction, cfg.c_z, cfg.c_hidden, cfg.dtype))
    out = B.trimul(z, M, p, direction)
    torch.cuda.synchronize()
    masked = np.where(m.numpy() == 0)[0]
    extra = masked[:4] if len(masked) else ()
    I = U.sample_indices(N, n_idx, seed, tile=256, extra=extra)
    J = U.sample_indices(N, n_idx, seed + 1, tile=256, extra=extra)
    ref = U.oracle_subgrid(z, M, p, direction, I, J)
    It, Jt = torch.as_tensor(I, device=DEV), torch.as_tensor(J, device=DEV)
    got = U.np64(out[It][:, Jt])
    e = U.assert_parity(got, ref, cfg.dtype, f"cfg{cfg.index} N={N} dir={direction} (sub-grid {n_idx}^2)")
    # masked pairs are exactly zero with the output mask on
    if len(masked):
        assert torch.all(out[int(masked[0])] == 0) and torch.all(out[:, int(masked[0])] == 0)
    return e


@pytest.mark.parametrize("direction", [OUT, INC])
def test_config2_bf16_n2048_chains(direction):
    run_subgrid(synth.CONFIGS[2], direction, 128, 11)


@pytest.mark.parametrize("direction", [OUT, INC])
def test_config3_bf16_n4096_headline(direction):
    run_subgrid(synth.CONFIGS[3], direction, 128, 12)


@pytest.mark.parametrize("direction", [OUT, INC])
def test_config4_bf16_n8192_single_call(direction):
    free, _ = torch.cuda.mem_get_info()
    if free < 100 * 2 ** 30:
        pytest.skip("needs ~85 GiB of free HBM")
    run_subgrid(synth.CONFIGS[4], direction, 128, 13)
    torch.cuda.empty_cache()


# ---------------------------------------------------------------- randomised sweep (full oracle)
def test_randomised_sweep_against_oracle():
    """Seeded sweep over sizes (multiples of 8 up to 320: partial tiles in every kernel), both
    directions, mask kinds (incl. a general non-symmetric pair mask and NULL), missing biases,
    output mask on / off, residual on / off, and input scale / offset."""
    import random
    from oracle import trimul_oracle as orc
    rnd = random.Random(20260314)
    cfg = synth.CONFIGS[1]
    for trial in range(12):
        N = 8 * rnd.randint(1, 40)
        d = rnd.randint(0, 1)
        mo, res = rnd.random() < 0.7, rnd.random() < 0.4
        mk = rnd.choice(["ones", "tail", "scatter", "none", "rand"])
        z, _, p = synth.make_inputs(cfg, d, "cpu", N=N)
        g = torch.Generator().manual_seed(trial)
        z = (z.float() * (0.2 + 3 * torch.rand(1, generator=g)) + torch.randn(1, generator=g)).to(torch.bfloat16)
        if mk == "none":
            M = None
        elif mk == "rand":
            M = (torch.rand(N, N, generator=g) > 0.3).to(torch.bfloat16)
        else:
            M = synth.pair_mask(synth.make_token_mask(mk, N, trial), "bf16")
        if rnd.random() < 0.3:
            p = dict(p)
            p[rnd.choice(["b_a", "b_g", "b_o", "b_b_gate"])] = None
        upd = orc.trimul(U.np64(z), None if M is None else U.np64(M), U.params64(p), d, mask_output=mo)
        ref = upd + (U.np64(z) if res else 0.0)
        out = B.trimul(z.to(DEV), None if M is None else M.to(DEV),
                       {k: (None if v is None else v.to(DEV)) for k, v in p.items()}, d,
                       mask_output=mo, residual=res)
        torch.cuda.synchronize()
        got = U.np64(out)
        what = f"trial {trial}: N={N} dir={d} mask={mk} mask_output={mo} residual={res}"
        assert np.all(np.isfinite(got)), what
        # north_star tolerance on the update; the residual form adds the rounding of z + update
        tol = U.TOL["bf16"]["max_over_rms"] * np.sqrt(np.mean(upd ** 2)) + \
            (2.0 ** -9 * np.abs(ref).max() if res else 0.0)
        assert np.abs(got - ref).max() <= tol, what
        assert np.linalg.norm(got - ref) <= U.TOL["bf16"]["rel_fro"] * np.linalg.norm(ref), what
