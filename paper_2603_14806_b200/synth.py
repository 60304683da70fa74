"""Seeded synthetic inputs for the triangle multiplicative update.

This module is the ONLY code shared by the CPU oracle's tests and the CUDA path.
It holds none of the method's arithmetic: it only draws random tensors with the
shapes / value distributions BASELINE.json's `configs` name (z ~ N(0,1); Linear
weights ~ N(0, 1/fan_in); biases ~ N(0, 0.02^2); LayerNorm gamma = 1 + 0.1 N(0,1),
beta = 0.1 N(0,1); non-zero output projection) and builds the token / pair masks
those configs describe.  Stand-ins for the paper's workloads (trained Boltz pair
activations at the token scales of PAPER.md Table 2 / Fig. 3) --
see DESIGN.md "Input recipe".

Values are drawn in fp32 and, for the bf16 configs, z / mask / the six weight
matrices are rounded to bf16 ONCE here; both the oracle and the GPU receive those
rounded values, so input quantisation is never charged to either side.
"""
from __future__ import annotations

import dataclasses
from typing import Dict, List, Optional

import torch

# tensor ids (mixed into the seed so every tensor has its own stream)
_TID = {
    "z": 1, "ln_in_gamma": 2, "ln_in_beta": 3,
    "w_a": 4, "b_a": 5, "w_a_gate": 6, "b_a_gate": 7,
    "w_b": 8, "b_b": 9, "w_b_gate": 10, "b_b_gate": 11,
    "w_g": 12, "b_g": 13, "ln_out_gamma": 14, "ln_out_beta": 15,
    "w_o": 16, "b_o": 17, "mask": 18,
}

PARAM_MATRICES = ("w_a", "w_a_gate", "w_b", "w_b_gate", "w_g", "w_o")
PARAM_VECTORS = ("ln_in_gamma", "ln_in_beta", "b_a", "b_a_gate", "b_b", "b_b_gate",
                 "b_g", "ln_out_gamma", "ln_out_beta", "b_o")


@dataclasses.dataclass(frozen=True)
class Config:
    """One BASELINE.json config (index = position in its `configs` list)."""
    index: int
    N: int
    dtype: str            # "f32" | "bf16"
    mask_kind: str        # "ones" | "tail" | "chains" | "scatter"
    seed: int
    c_z: int = 128
    c_hidden: int = 128


CONFIGS: List[Config] = [
    Config(0, 64, "f32", "ones", 1000),
    Config(1, 512, "bf16", "tail", 1001),
    Config(2, 2048, "bf16", "chains", 1002),
    Config(3, 4096, "bf16", "ones", 1003),
    Config(4, 8192, "bf16", "scatter", 1004),
]


def _gen(seed: int, name: str, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(int(seed) * 1000003 + _TID[name])
    return g


def _tdtype(dtype: str) -> torch.dtype:
    if dtype == "f32":
        return torch.float32
    if dtype == "bf16":
        return torch.bfloat16
    raise ValueError(f"dtype must be 'f32' or 'bf16', got {dtype!r}")


def make_params(seed: int, c_z: int = 128, c_hidden: int = 128, dtype: str = "bf16",
                device="cpu") -> Dict[str, torch.Tensor]:
    """Parameter set of one triangle-multiplication layer.

    Weight matrices are torch-Linear layout [out_features, in_features] in `dtype`
    (already rounded); LayerNorm affine parameters and biases are fp32.
    """
    td = _tdtype(dtype)
    shapes = {
        "w_a": (c_hidden, c_z), "w_a_gate": (c_hidden, c_z),
        "w_b": (c_hidden, c_z), "w_b_gate": (c_hidden, c_z),
        "w_g": (c_z, c_z), "w_o": (c_z, c_hidden),
    }
    p: Dict[str, torch.Tensor] = {}
    for name, (fo, fi) in shapes.items():
        w = torch.randn(fo, fi, generator=_gen(seed, name, "cpu"), dtype=torch.float32)
        p[name] = (w * (fi ** -0.5)).to(td).to(device)
    bias_len = {"b_a": c_hidden, "b_a_gate": c_hidden, "b_b": c_hidden,
                "b_b_gate": c_hidden, "b_g": c_z, "b_o": c_z}
    for name, n in bias_len.items():
        p[name] = (0.02 * torch.randn(n, generator=_gen(seed, name, "cpu"),
                                      dtype=torch.float32)).to(device)
    for pre, n in (("ln_in", c_z), ("ln_out", c_hidden)):
        p[pre + "_gamma"] = (1.0 + 0.1 * torch.randn(
            n, generator=_gen(seed, pre + "_gamma", "cpu"), dtype=torch.float32)).to(device)
        p[pre + "_beta"] = (0.1 * torch.randn(
            n, generator=_gen(seed, pre + "_beta", "cpu"), dtype=torch.float32)).to(device)
    return p


def make_z(seed: int, N: int, c_z: int = 128, dtype: str = "bf16", device="cpu",
           chunk_rows: int = 256) -> torch.Tensor:
    """Pair representation z[N, N, c_z] ~ N(0,1), drawn row-chunk by row-chunk so the
    fp32 staging never exceeds chunk_rows*N*c_z*4 bytes (N=8192 is 16 GiB in bf16)."""
    td = _tdtype(dtype)
    z = torch.empty(N, N, c_z, dtype=td, device=device)
    g = _gen(seed, "z", device)
    for r0 in range(0, N, chunk_rows):
        r1 = min(N, r0 + chunk_rows)
        z[r0:r1] = torch.randn(r1 - r0, N, c_z, generator=g, dtype=torch.float32,
                               device=device).to(td)
    return z


def make_token_mask(kind: str, N: int, seed: int) -> torch.Tensor:
    """Token mask m[N] (fp32 0/1) for the four patterns BASELINE.json's configs use."""
    m = torch.ones(N, dtype=torch.float32)
    g = _gen(seed, "mask", "cpu")
    if kind == "ones":
        pass
    elif kind == "tail":            # config 1: last 10% of tokens are padding
        m[N - (N // 10):] = 0.0
    elif kind == "chains":          # config 2: 4 chains summing to 1900 of 2048, rest padding
        valid = (N * 1900) // 2048
        m[valid:] = 0.0
    elif kind == "scatter":         # config 4: a random 5% of tokens zeroed
        k = int(round(0.05 * N))
        idx = torch.randperm(N, generator=g)[:k]
        m[idx] = 0.0
    else:
        raise ValueError(kind)
    return m


def chain_lengths(N: int, seed: int, n_chains: int = 4, min_len: int = 50) -> List[int]:
    """Config 2's seeded composition of the valid tokens into `n_chains` chains (each >=
    min_len).  Chain boundaries do not enter the mask (padding is at the end); they are
    used by the chain-permutation equivariance test."""
    valid = (N * 1900) // 2048
    g = _gen(seed, "mask", "cpu")
    free = valid - n_chains * min_len
    cuts = torch.sort(torch.randint(0, free + 1, (n_chains - 1,), generator=g)).values.tolist()
    edges = [0] + cuts + [free]
    return [min_len + (edges[i + 1] - edges[i]) for i in range(n_chains)]


def pair_mask(m: torch.Tensor, dtype: str = "bf16", device="cpu") -> torch.Tensor:
    """Pair mask M[N, N] = m_i * m_j in the tensor dtype (the library's ABI takes a PAIR mask)."""
    M = m[:, None] * m[None, :]
    return M.to(_tdtype(dtype)).to(device)


def make_inputs(cfg: Config, direction: int, device="cpu", N: Optional[int] = None):
    """(z, M, params) of one BASELINE config; the two directions are separate layers and
    get different seeded parameter sets (same z)."""
    n = cfg.N if N is None else N
    z = make_z(cfg.seed, n, cfg.c_z, cfg.dtype, device)
    m = make_token_mask(cfg.mask_kind, n, cfg.seed)
    M = pair_mask(m, cfg.dtype, device)
    p = make_params(cfg.seed * 2 + int(direction), cfg.c_z, cfg.c_hidden, cfg.dtype, device)
    return z, M, p


def make_z_slices(seed: int, rows: int, N: int, c_z: int = 128, dtype: str = "bf16"):
    """The slices of a z ~ N(0,1) pair tensor that a rows x rows sub-grid evaluation touches:
    (z_a [rows, N, c_z], z_b [rows, N, c_z], z_ij [rows, rows, c_z]) -- same distribution as make_z,
    drawn directly so the bounded CPU-baseline sample never materialises the N x N tensor."""
    td = _tdtype(dtype)
    g = _gen(seed, "z", "cpu")
    za = torch.randn(rows, N, c_z, generator=g, dtype=torch.float32).to(td)
    zb = torch.randn(rows, N, c_z, generator=g, dtype=torch.float32).to(td)
    zij = torch.randn(rows, rows, c_z, generator=g, dtype=torch.float32).to(td)
    return za, zb, zij
