"""ctypes binding of libfoldcp_trimul.so -- argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI (include/foldcp_trimul.h);
PyTorch is used for device memory and streams.  There is NO CPU fallback: if the shared library
is missing or a call fails, this raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Dict, Optional

import torch

OUTGOING = 0
INCOMING = 1
F32 = 0
BF16 = 1
BF16_F16AB = 2     # foldcp_trimul_contract only: a, b fp16 (as the project stage writes them), o bf16
BF16_F16ALL = 3    # foldcp_trimul_contract only: a, b fp16; o fp16 scaled by o_scale(N) (the fused form)

_LIB_NAME = "libfoldcp_trimul.so"
_lib = None

EXPORTS = (
    "foldcp_trimul", "foldcp_trimul_batched", "foldcp_trimul_workspace_bytes", "foldcp_trimul_project",
    "foldcp_trimul_contract", "foldcp_trimul_contract_backward", "foldcp_trimul_finalize", "foldcp_trimul_launches_per_call",
    "foldcp_trimul_backward", "foldcp_trimul_backward_workspace_bytes", "foldcp_trimul_contract_blocks",
    "foldcp_trimul_project_stats", "foldcp_trimul_finalize_fused", "foldcp_trimul_o_scale",
    "foldcp_triattn", "foldcp_triattn_workspace_bytes",
    "foldcp_trimul_static", "foldcp_trimul_static_max_n", "foldcp_trimul_static_workspace_bytes",
    "foldcp_status_string", "foldcp_version",
)


class FoldcpError(RuntimeError):
    def __init__(self, status: int, what: str):
        self.status = status
        super().__init__(f"{what}: status {status} ({status_string(status)})")


class _Params(ctypes.Structure):
    _fields_ = [
        ("struct_size", ctypes.c_uint32), ("dtype", ctypes.c_int32),
        ("ln_eps", ctypes.c_float), ("mask_output", ctypes.c_int32),
        ("add_residual", ctypes.c_int32), ("reserved0", ctypes.c_int32),
        ("ln_in_gamma", ctypes.c_void_p), ("ln_in_beta", ctypes.c_void_p),
        ("w_a", ctypes.c_void_p), ("w_a_gate", ctypes.c_void_p),
        ("w_b", ctypes.c_void_p), ("w_b_gate", ctypes.c_void_p),
        ("b_a", ctypes.c_void_p), ("b_a_gate", ctypes.c_void_p),
        ("b_b", ctypes.c_void_p), ("b_b_gate", ctypes.c_void_p),
        ("w_g", ctypes.c_void_p), ("b_g", ctypes.c_void_p),
        ("ln_out_gamma", ctypes.c_void_p), ("ln_out_beta", ctypes.c_void_p),
        ("w_o", ctypes.c_void_p), ("b_o", ctypes.c_void_p),
        ("workspace", ctypes.c_void_p), ("workspace_bytes", ctypes.c_size_t),
    ]


PARAM_NAMES = ("ln_in_gamma", "ln_in_beta", "w_a", "w_a_gate", "w_b", "w_b_gate", "b_a", "b_a_gate",
               "b_b", "b_b_gate", "w_g", "b_g", "ln_out_gamma", "ln_out_beta", "w_o", "b_o")


class _TriAttnParams(ctypes.Structure):
    _fields_ = [
        ("struct_size", ctypes.c_uint32), ("dtype", ctypes.c_int32), ("ln_eps", ctypes.c_float),
        ("n_heads", ctypes.c_int32),
        ("ln_gamma", ctypes.c_void_p), ("ln_beta", ctypes.c_void_p),
        ("w_q", ctypes.c_void_p), ("w_k", ctypes.c_void_p), ("w_v", ctypes.c_void_p),
        ("w_g", ctypes.c_void_p), ("w_t", ctypes.c_void_p), ("w_o", ctypes.c_void_p),
        ("workspace", ctypes.c_void_p), ("workspace_bytes", ctypes.c_size_t),
    ]


TRIATTN_STARTING = 0
TRIATTN_ENDING = 1


class _Grads(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_uint32), ("reserved0", ctypes.c_uint32)] + \
               [(name, ctypes.c_void_p) for name in PARAM_NAMES]


def lib_path() -> str:
    return os.path.join(os.path.dirname(os.path.abspath(__file__)), _LIB_NAME)


def load() -> ctypes.CDLL:
    """Load the shared library (raises if it has not been built: no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise RuntimeError(
            f"{path} is missing: build it with `python -m paper_2603_14806_b200.build` "
            "(there is no CPU fallback)")
    lib = ctypes.CDLL(path)
    vp, ci = ctypes.c_void_p, ctypes.c_int
    lib.foldcp_trimul.restype = ci
    lib.foldcp_trimul.argtypes = [vp, vp, ctypes.POINTER(_Params), ci, ci, ci, ci, vp, vp]
    lib.foldcp_trimul_batched.restype = ci
    lib.foldcp_trimul_batched.argtypes = [vp, vp, ctypes.POINTER(_Params), ci, ci, ci, ci, ci, vp, vp]
    lib.foldcp_trimul_workspace_bytes.restype = ctypes.c_size_t
    lib.foldcp_trimul_workspace_bytes.argtypes = [ci, ci, ci, ci]
    lib.foldcp_trimul_project.restype = ci
    lib.foldcp_trimul_project.argtypes = [vp, vp, ctypes.POINTER(_Params), ci, ci, ci, vp, vp, vp, vp]
    lib.foldcp_trimul_contract_backward.restype = ci
    lib.foldcp_trimul_contract_backward.argtypes = [vp, vp, vp, ci, ci, ci, ci, vp, vp, vp, vp]
    lib.foldcp_trimul_contract.restype = ci
    lib.foldcp_trimul_contract.argtypes = [vp, vp, ci, ci, ci, ci, vp, vp, vp]
    lib.foldcp_trimul_finalize.restype = ci
    lib.foldcp_trimul_finalize.argtypes = [vp, vp, vp, ctypes.POINTER(_Params), ci, ci, ci, vp, vp]
    lib.foldcp_trimul_project_stats.restype = ci
    lib.foldcp_trimul_project_stats.argtypes = [vp, vp, ctypes.POINTER(_Params), ci, ci, ci, vp, vp, vp, vp, vp]
    lib.foldcp_trimul_finalize_fused.restype = ci
    lib.foldcp_trimul_finalize_fused.argtypes = [vp, vp, vp, vp, ctypes.POINTER(_Params), ci, ci, ci, vp, vp]
    lib.foldcp_trimul_o_scale.restype = ctypes.c_float
    lib.foldcp_trimul_o_scale.argtypes = [ci]
    lib.foldcp_trimul_contract_blocks.restype = ci
    lib.foldcp_trimul_contract_blocks.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(vp), ci, ci, ci, ci, ci,
                                                  vp, vp, vp]
    lib.foldcp_trimul_backward.restype = ci
    lib.foldcp_trimul_backward.argtypes = [vp, vp, vp, ctypes.POINTER(_Params), ci, ci, ci, ci, vp,
                                           ctypes.POINTER(_Grads), vp]
    lib.foldcp_trimul_backward_workspace_bytes.restype = ctypes.c_size_t
    lib.foldcp_trimul_backward_workspace_bytes.argtypes = [ci, ci, ci, ci]
    lib.foldcp_trimul_launches_per_call.restype = ci
    lib.foldcp_trimul_launches_per_call.argtypes = [ci]
    lib.foldcp_triattn.restype = ci
    lib.foldcp_triattn.argtypes = [vp, vp, ctypes.POINTER(_TriAttnParams), ci, ci, ci, vp, vp]
    lib.foldcp_triattn_workspace_bytes.restype = ctypes.c_size_t
    lib.foldcp_triattn_workspace_bytes.argtypes = [ci, ci, ci, ci]
    lib.foldcp_trimul_static.restype = ci
    lib.foldcp_trimul_static.argtypes = [vp, vp, ctypes.POINTER(_Params), ci, ci, ci, ci, vp, vp]
    lib.foldcp_trimul_static_max_n.restype = ci
    lib.foldcp_trimul_static_max_n.argtypes = [ci, ci, ci]
    lib.foldcp_trimul_static_workspace_bytes.restype = ctypes.c_size_t
    lib.foldcp_trimul_static_workspace_bytes.argtypes = []
    lib.foldcp_status_string.restype = ctypes.c_char_p
    lib.foldcp_status_string.argtypes = [ci]
    lib.foldcp_version.restype = ci
    lib.foldcp_version.argtypes = []
    _lib = lib
    return lib


def status_string(status: int) -> str:
    return load().foldcp_status_string(int(status)).decode()


def version() -> int:
    return load().foldcp_version()


def dtype_code(t: torch.Tensor) -> int:
    if t.dtype == torch.float32:
        return F32
    if t.dtype == torch.bfloat16:
        return BF16
    raise TypeError(f"unsupported dtype {t.dtype}: z must be float32 or bfloat16")


def workspace_bytes(N: int, c_z: int = 128, c_hidden: int = 128, dtype: int = BF16) -> int:
    return int(load().foldcp_trimul_workspace_bytes(N, c_z, c_hidden, dtype))


def backward_workspace_bytes(N: int, c_z: int = 128, c_hidden: int = 128, dtype: int = BF16) -> int:
    return int(load().foldcp_trimul_backward_workspace_bytes(N, c_z, c_hidden, dtype))


def launches_per_call(dtype: int = BF16) -> int:
    return int(load().foldcp_trimul_launches_per_call(dtype))


def _ptr(t: Optional[torch.Tensor]) -> Optional[int]:
    return None if t is None else t.data_ptr()


SCHED_SCRATCH_BYTES = 256      # FOLDCP_SCHED_SCRATCH_BYTES


def stage_scratch(device) -> torch.Tensor:
    """The `scratch` argument of the stage entry points: tile counters of one call (the library
    zeroes it on the stream).  Allocated per call on the current stream: torch's caching allocator
    only hands the block out again to work ordered after this call on the same stream."""
    return torch.empty(SCHED_SCRATCH_BYTES, dtype=torch.uint8, device=device)


_MATRICES = ("w_a", "w_a_gate", "w_b", "w_b_gate", "w_g", "w_o")


def _check_tensors(z: torch.Tensor, p: Dict[str, Optional[torch.Tensor]], others=()) -> None:
    """The C ABI sees raw pointers: dtype / device / contiguity mismatches would be silent garbage,
    so they are rejected here.  The library launches on the CURRENT device and stream."""
    if not z.is_cuda:
        raise ValueError("tensors must be CUDA tensors (no CPU fallback)")
    if z.device.index != torch.cuda.current_device():
        raise ValueError(f"z is on {z.device} but the current CUDA device is "
                         f"cuda:{torch.cuda.current_device()} (use torch.cuda.device(...))")
    for name, t in list(p.items()) + [(f"arg{i}", t) for i, t in enumerate(others)]:
        if t is None:
            continue
        if t.device != z.device:
            raise ValueError(f"{name} is on {t.device}, z on {z.device}")
        if not t.is_contiguous():
            raise ValueError(f"{name} must be contiguous")
        if name in _MATRICES:
            if t.dtype != z.dtype:
                raise TypeError(f"{name} has dtype {t.dtype}; weight matrices must match z ({z.dtype})")
        elif name in p and t.dtype != torch.float32:
            raise TypeError(f"{name} has dtype {t.dtype}; LayerNorm parameters and biases are float32")


def make_params(p: Dict[str, Optional[torch.Tensor]], dtype: int, eps: float = 1e-5,
                mask_output: bool = True, workspace: Optional[torch.Tensor] = None,
                residual: bool = False) -> _Params:
    """Fill the C struct from a dict of device tensors (names of synth.make_params)."""
    s = _Params()
    s.struct_size = ctypes.sizeof(_Params)
    s.dtype = dtype
    s.ln_eps = eps
    s.mask_output = 1 if mask_output else 0
    s.add_residual = 1 if residual else 0
    s.reserved0 = 0
    for name in ("ln_in_gamma", "ln_in_beta", "w_a", "w_a_gate", "w_b", "w_b_gate", "b_a",
                 "b_a_gate", "b_b", "b_b_gate", "w_g", "b_g", "ln_out_gamma", "ln_out_beta",
                 "w_o", "b_o"):
        setattr(s, name, _ptr(p.get(name)))
    if workspace is not None:
        s.workspace = workspace.data_ptr()
        s.workspace_bytes = workspace.numel() * workspace.element_size()
    return s


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def trimul(z: torch.Tensor, mask: Optional[torch.Tensor], p: Dict[str, torch.Tensor],
           direction: int, out: Optional[torch.Tensor] = None,
           workspace: Optional[torch.Tensor] = None, eps: float = 1e-5,
           mask_output: bool = True, residual: bool = False) -> torch.Tensor:
    """One forward triangle multiplicative update on the current CUDA stream (asynchronous).

    z [N, N, c_z] and mask [N, N] (or None) are CUDA tensors of the same dtype (fp32 / bf16);
    a leading batch dimension (z [B, N, N, c_z], mask [B, N, N]) goes through
    foldcp_trimul_batched.  `residual=True` returns z + update (the paper's "z +=" form).
    `workspace` (uint8, >= workspace_bytes(N)) and `out` are allocated here if not given.
    """
    lib = load()
    _check_tensors(z, p, (mask, out, workspace))
    batch = None
    if z.dim() == 4:
        batch = z.shape[0]
        assert z.shape[1] == z.shape[2] and z.is_contiguous()
        N, c_z = z.shape[1], z.shape[3]
    else:
        assert z.dim() == 3 and z.shape[0] == z.shape[1] and z.is_contiguous()
        N, c_z = z.shape[0], z.shape[2]
    c_hidden = p["w_a"].shape[0]
    dt = dtype_code(z)
    if mask is not None:
        assert mask.dtype == z.dtype and mask.is_contiguous() and mask.shape == z.shape[:-1]
    if workspace is None:
        workspace = torch.empty(max(workspace_bytes(N, c_z, c_hidden, dt), 1), dtype=torch.uint8,
                                device=z.device)
    if out is None:
        out = torch.empty_like(z)
    s = make_params(p, dt, eps, mask_output, workspace, residual)
    if batch is None:
        st = lib.foldcp_trimul(z.data_ptr(), _ptr(mask), ctypes.byref(s), N, c_z, c_hidden,
                               int(direction), out.data_ptr(), _stream())
    else:
        st = lib.foldcp_trimul_batched(z.data_ptr(), _ptr(mask), ctypes.byref(s), batch, N, c_z,
                                       c_hidden, int(direction), out.data_ptr(), _stream())
    if st != 0:
        raise FoldcpError(st, "foldcp_trimul")
    return out


def static_max_n(dtype: int, c_z: int = 128, c_hidden: int = 128) -> int:
    """Largest N trimul_static accepts for this dtype code (foldcp_trimul_static_max_n)."""
    return load().foldcp_trimul_static_max_n(c_z, c_hidden, int(dtype))


def static_workspace_bytes() -> int:
    return load().foldcp_trimul_static_workspace_bytes()


def trimul_static(z: torch.Tensor, mask: Optional[torch.Tensor], p: Dict[str, torch.Tensor],
                  direction: int, out: torch.Tensor, eps: float = 1e-5,
                  mask_output: bool = True, residual: bool = False) -> torch.Tensor:
    """foldcp_trimul_static: trimul() with the scratch in the library's static device array.

    Allocates nothing (neither here nor in the library): `out` must be given, no workspace is
    passed.  N <= static_max_n(dtype); beyond it FoldcpError with FOLDCP_ERR_STATIC_LIMIT (8).
    All calls on a device share the one array: calls that may overlap on the GPU race.
    """
    lib = load()
    _check_tensors(z, p, (mask, out))
    assert z.dim() == 3 and z.shape[0] == z.shape[1] and z.is_contiguous()
    assert out.shape == z.shape and out.dtype == z.dtype and out.is_contiguous()
    N, c_z = z.shape[0], z.shape[2]
    c_hidden = p["w_a"].shape[0]
    if mask is not None:
        assert mask.dtype == z.dtype and mask.is_contiguous() and mask.shape == z.shape[:-1]
    s = make_params(p, dtype_code(z), eps, mask_output, None, residual)
    st = lib.foldcp_trimul_static(z.data_ptr(), _ptr(mask), ctypes.byref(s), N, c_z, c_hidden,
                                  int(direction), out.data_ptr(), _stream())
    if st != 0:
        raise FoldcpError(st, "foldcp_trimul_static")
    return out


def project(z, mask, p, eps: float = 1e-5):
    """Stage a1+a2: returns (a, b), each [c_hidden, N, N] channel-major."""
    lib = load()
    N, c_z = z.shape[0], z.shape[2]
    c_hidden = p["w_a"].shape[0]
    _check_tensors(z, p, (mask,))
    # bf16 mode stores the intermediates a, b as fp16 (include/foldcp_trimul.h, numeric preconditions)
    ab_dtype = torch.float16 if z.dtype == torch.bfloat16 else z.dtype
    a = torch.empty(c_hidden, N, N, dtype=ab_dtype, device=z.device)
    b = torch.empty_like(a)
    s = make_params(p, dtype_code(z), eps)
    st = lib.foldcp_trimul_project(z.data_ptr(), _ptr(mask), ctypes.byref(s), N, c_z, c_hidden,
                                   a.data_ptr(), b.data_ptr(), stage_scratch(z.device).data_ptr(),
                                   _stream())
    if st != 0:
        raise FoldcpError(st, "foldcp_trimul_project")
    return a, b


def o_scale(N: int) -> float:
    """The power of two by which the fused call scales o between its last two kernels."""
    return float(load().foldcp_trimul_o_scale(int(N)))


def project_stats(z, mask, p, eps: float = 1e-5):
    """Stage a1+a2 in the fused form (bf16 mode): returns (a, b, z_stats) with z_stats [N, N, 2] fp32 =
    (mean, rstd) of LayerNorm(z) per pair."""
    lib = load()
    N, c_z = z.shape[0], z.shape[2]
    c_hidden = p["w_a"].shape[0]
    _check_tensors(z, p, (mask,))
    a = torch.empty(c_hidden, N, N, dtype=torch.float16, device=z.device)
    b = torch.empty_like(a)
    stats = torch.empty(N, N, 2, dtype=torch.float32, device=z.device)
    s = make_params(p, dtype_code(z), eps)
    st = lib.foldcp_trimul_project_stats(z.data_ptr(), _ptr(mask), ctypes.byref(s), N, c_z, c_hidden,
                                         a.data_ptr(), b.data_ptr(), stats.data_ptr(),
                                         stage_scratch(z.device).data_ptr(), _stream())
    if st != 0:
        raise FoldcpError(st, "foldcp_trimul_project_stats")
    return a, b, stats


def finalize_fused(o, z, z_stats, mask, p, eps: float = 1e-5, mask_output: bool = True,
                   residual: bool = False, out: Optional[torch.Tensor] = None):
    """Stage a3+a5 in the fused form: o [c, N, N] fp16 scaled by o_scale(N); z_stats from
    project_stats (or None: recomputed)."""
    lib = load()
    N, c_z = z.shape[0], z.shape[2]
    c_hidden = o.shape[0]
    assert o.dtype == torch.float16
    if out is None:
        out = torch.empty_like(z)
    _check_tensors(z, p, (o, mask, out, z_stats))
    s = make_params(p, dtype_code(z), eps, mask_output, None, residual)
    st = lib.foldcp_trimul_finalize_fused(o.data_ptr(), z.data_ptr(), _ptr(z_stats), _ptr(mask),
                                          ctypes.byref(s), N, c_z, c_hidden, out.data_ptr(), _stream())
    if st != 0:
        raise FoldcpError(st, "foldcp_trimul_finalize_fused")
    return out


def contract(a: torch.Tensor, b: torch.Tensor, direction: int,
             o: Optional[torch.Tensor] = None, fused_o: bool = False) -> torch.Tensor:
    """Stage a4 (Eq. 2-3): a, b [c, N, N] channel-major -> o [c, N, N].  a, b may be fp32, bf16 or
    fp16 (the project stage's output in bf16 mode; o is then bf16)."""
    lib = load()
    c, N = a.shape[0], a.shape[1]
    assert a.dtype == b.dtype
    if a.dtype == torch.float16:
        code, o_dtype = (BF16_F16ALL, torch.float16) if fused_o else (BF16_F16AB, torch.bfloat16)
    else:
        assert not fused_o
        code, o_dtype = dtype_code(a), a.dtype
    if o is None:
        o = torch.empty(a.shape, dtype=o_dtype, device=a.device)
    _check_tensors(a, {}, (b, o))
    st = lib.foldcp_trimul_contract(a.data_ptr(), b.data_ptr(), N, c, code,
                                    int(direction), o.data_ptr(),
                                    stage_scratch(a.device).data_ptr(), _stream())
    if st != 0:
        raise FoldcpError(st, "foldcp_trimul_contract")
    return o


def contract_blocks(a_blocks, b_blocks, direction: int, o_block: Optional[torch.Tensor] = None) -> torch.Tensor:
    """Blocked (Cannon) contraction: o_block = sum_q contraction(a_blocks[q], b_blocks[q]); every
    block a contiguous [c, nb, nb] channel-major tensor (fp32 / bf16 / fp16 like `contract`)."""
    lib = load()
    a0 = a_blocks[0]
    c, nb = a0.shape[0], a0.shape[1]
    assert len(a_blocks) == len(b_blocks) >= 1
    for t in list(a_blocks) + list(b_blocks):
        assert t.shape == a0.shape and t.dtype == a0.dtype
    if a0.dtype == torch.float16:
        code, o_dtype = BF16_F16AB, torch.bfloat16
    else:
        code, o_dtype = dtype_code(a0), a0.dtype
    if o_block is None:
        o_block = torch.empty(a0.shape, dtype=o_dtype, device=a0.device)
    _check_tensors(a0, {}, tuple(a_blocks) + tuple(b_blocks) + (o_block,))
    n = len(a_blocks)
    pa = (ctypes.c_void_p * n)(*[t.data_ptr() for t in a_blocks])
    pb = (ctypes.c_void_p * n)(*[t.data_ptr() for t in b_blocks])
    st = lib.foldcp_trimul_contract_blocks(pa, pb, n, nb, c, code, int(direction), o_block.data_ptr(),
                                           stage_scratch(a0.device).data_ptr(), _stream())
    if st != 0:
        raise FoldcpError(st, "foldcp_trimul_contract_blocks")
    return o_block


def contract_backward(d_o: torch.Tensor, a: torch.Tensor, b: torch.Tensor, direction: int):
    """Backward of stage a4: returns (d_a, d_b), each [c, N, N] channel-major."""
    lib = load()
    c, N = a.shape[0], a.shape[1]
    d_a, d_b = torch.empty_like(a), torch.empty_like(b)
    st = lib.foldcp_trimul_contract_backward(d_o.data_ptr(), a.data_ptr(), b.data_ptr(), N, c,
                                             dtype_code(a), int(direction), d_a.data_ptr(),
                                             d_b.data_ptr(), stage_scratch(a.device).data_ptr(),
                                             _stream())
    if st != 0:
        raise FoldcpError(st, "foldcp_trimul_contract_backward")
    return d_a, d_b


def finalize(o, z, mask, p, eps: float = 1e-5, mask_output: bool = True,
             out: Optional[torch.Tensor] = None):
    """Stage a3+a5: LayerNorm(o) + output projection + sigmoid gate + mask -> out [N, N, c_z]."""
    lib = load()
    N, c_z = z.shape[0], z.shape[2]
    c_hidden = o.shape[0]
    if out is None:
        out = torch.empty_like(z)
    _check_tensors(z, p, (o, mask, out))
    s = make_params(p, dtype_code(z), eps, mask_output)
    st = lib.foldcp_trimul_finalize(o.data_ptr(), z.data_ptr(), _ptr(mask), ctypes.byref(s), N,
                                    c_z, c_hidden, out.data_ptr(), _stream())
    if st != 0:
        raise FoldcpError(st, "foldcp_trimul_finalize")
    return out


def trimul_backward(d_out: torch.Tensor, z: torch.Tensor, mask: Optional[torch.Tensor],
                    p: Dict[str, Optional[torch.Tensor]], direction: int, eps: float = 1e-5,
                    mask_output: bool = True, residual: bool = False,
                    workspace: Optional[torch.Tensor] = None):
    """Full backward of one trimul call: returns (d_z, grads) with grads a dict of fp32 tensors, one
    per parameter present in `p` (same shapes).  Asynchronous on the current stream."""
    lib = load()
    _check_tensors(z, p, (d_out, mask, workspace))
    assert z.dim() == 3 and z.shape[0] == z.shape[1] and d_out.shape == z.shape and d_out.dtype == z.dtype
    N, c_z = z.shape[0], z.shape[2]
    c_hidden = p["w_a"].shape[0]
    dt = dtype_code(z)
    if workspace is None:
        workspace = torch.empty(max(backward_workspace_bytes(N, c_z, c_hidden, dt), 1),
                                dtype=torch.uint8, device=z.device)
    s = make_params(p, dt, eps, mask_output, workspace, residual)
    d_z = torch.empty_like(z)
    grads = {k: torch.empty(v.shape, dtype=torch.float32, device=z.device)
             for k, v in p.items() if v is not None}
    g = _Grads()
    g.struct_size = ctypes.sizeof(_Grads)
    g.reserved0 = 0
    for name in PARAM_NAMES:
        setattr(g, name, _ptr(grads.get(name)))
    st = lib.foldcp_trimul_backward(d_out.data_ptr(), z.data_ptr(), _ptr(mask), ctypes.byref(s), N,
                                    c_z, c_hidden, int(direction), d_z.data_ptr(), ctypes.byref(g),
                                    _stream())
    if st != 0:
        raise FoldcpError(st, "foldcp_trimul_backward")
    return d_z, grads


def triattn_workspace_bytes(N: int, c_z: int = 128, n_heads: int = 4, dtype: int = BF16) -> int:
    return int(load().foldcp_triattn_workspace_bytes(N, c_z, n_heads, dtype))


def triattn(z: torch.Tensor, mask: Optional[torch.Tensor], p: Dict[str, torch.Tensor], node: int,
            n_heads: int = 4, eps: float = 1e-5, out: Optional[torch.Tensor] = None,
            workspace: Optional[torch.Tensor] = None) -> torch.Tensor:
    """Triangle attention (include/foldcp_triattn.h), starting (rows) or ending (columns) node, on the
    current CUDA stream.  p: ln_gamma, ln_beta (fp32), w_q, w_k, w_v, w_g [H*c, c_z], w_t [H, c_z],
    w_o [c_z, H*c] in z's dtype."""
    lib = load()
    assert z.dim() == 3 and z.shape[0] == z.shape[1] and z.is_contiguous() and z.is_cuda
    if z.device.index != torch.cuda.current_device():
        raise ValueError("z is not on the current CUDA device")
    N, c_z = z.shape[0], z.shape[2]
    dt = dtype_code(z)
    for name in ("w_q", "w_k", "w_v", "w_g", "w_t", "w_o"):
        t = p[name]
        if t.dtype != z.dtype or t.device != z.device or not t.is_contiguous():
            raise TypeError(f"{name}: dtype / device / contiguity must match z")
    for name in ("ln_gamma", "ln_beta"):
        if p[name].dtype != torch.float32 or p[name].device != z.device:
            raise TypeError(f"{name} must be float32 on z's device")
    if mask is not None:
        assert mask.dtype == z.dtype and mask.is_contiguous() and mask.shape == z.shape[:-1]
    if workspace is None:
        workspace = torch.empty(max(triattn_workspace_bytes(N, c_z, n_heads, dt), 1), dtype=torch.uint8,
                                device=z.device)
    if out is None:
        out = torch.empty_like(z)
    s = _TriAttnParams()
    s.struct_size = ctypes.sizeof(_TriAttnParams)
    s.dtype = dt
    s.ln_eps = eps
    s.n_heads = n_heads
    for name in ("ln_gamma", "ln_beta", "w_q", "w_k", "w_v", "w_g", "w_t", "w_o"):
        setattr(s, name, p[name].data_ptr())
    s.workspace = workspace.data_ptr()
    s.workspace_bytes = workspace.numel()
    st = lib.foldcp_triattn(z.data_ptr(), _ptr(mask), ctypes.byref(s), N, c_z, int(node), out.data_ptr(),
                            _stream())
    if st != 0:
        raise FoldcpError(st, "foldcp_triattn")
    return out
