"""ctypes marshalling for libmfsdp.so.  Same names as include/mfsdp.h; no arithmetic of the method lives here."""
import ctypes as C
import os
from dataclasses import dataclass

PKG = os.path.dirname(os.path.abspath(__file__))

BF16, F32 = 0, 1
ROLE_MATRIX, ROLE_TAIL = 0, 1
POLICY_ROLE_GREEDY, POLICY_SCOPE_GREEDY, POLICY_COST_AWARE = 0, 1, 2
METRIC_NUMEL, METRIC_NS_FLOPS = 0, 1
SCALE_MATCH_RMS_ADAMW, SCALE_ORIGINAL, SCALE_NONE = 0, 1, 2
NS_BF16, NS_FP32 = 0, 1
STEP_KEEP_O = 1
SHAMPOO_KEEP_D = 1
OK, EINVAL, ECAP, ELAYOUT, EARCH, ECUDA, ECACHE, ETOOBIG = 0, -1, -2, -3, -4, -5, -6, -7


class Param(C.Structure):            # mfsdp_param_t
    _fields_ = [("block_id", C.c_uint32), ("ndim", C.c_uint32), ("rows", C.c_uint32), ("cols", C.c_uint32),
                ("dtype", C.c_uint32), ("flags", C.c_uint32)]


class Desc(C.Structure):             # mfsdp_desc_t
    _fields_ = [("role", C.c_uint32), ("param_id", C.c_uint32), ("block_id", C.c_uint32), ("rows", C.c_uint32),
                ("cols", C.c_uint32), ("dtype", C.c_uint32), ("flags", C.c_uint32), ("reserved", C.c_uint32),
                ("elem_off", C.c_uint64)]

    def as_dict(self):
        return dict(role=self.role, param_id=self.param_id, block_id=self.block_id, rows=self.rows, cols=self.cols,
                    dtype=self.dtype, flags=self.flags, elem_off=self.elem_off)


class MuonHParams(C.Structure):      # mfsdp_muon_hparams_t
    _fields_ = [("lr", C.c_double), ("weight_decay", C.c_double), ("momentum", C.c_double), ("a", C.c_double),
                ("b", C.c_double), ("c", C.c_double), ("eps", C.c_double), ("nesterov", C.c_int32),
                ("ns_steps", C.c_int32), ("scale_mode", C.c_int32), ("precision", C.c_int32),
                ("flags", C.c_uint32), ("reserved", C.c_uint32)]

    def __init__(self, lr=0.02, weight_decay=0.01, momentum=0.95, a=3.4445, b=-4.7750, c=2.0315, eps=1e-7,
                 nesterov=1, ns_steps=5, scale_mode=SCALE_MATCH_RMS_ADAMW, precision=NS_BF16, flags=0):
        super().__init__(lr, weight_decay, momentum, a, b, c, eps, int(nesterov), ns_steps, scale_mode, precision,
                         flags, 0)


class AdamWHParams(C.Structure):     # mfsdp_adamw_hparams_t
    _fields_ = [("lr", C.c_double), ("beta1", C.c_double), ("beta2", C.c_double), ("eps", C.c_double),
                ("weight_decay", C.c_double), ("step", C.c_int64)]

    def __init__(self, lr=1e-3, beta1=0.9, beta2=0.95, eps=1e-8, weight_decay=0.01, step=1):
        super().__init__(lr, beta1, beta2, eps, weight_decay, step)


class ShampooHParams(C.Structure):   # mfsdp_shampoo_hparams_t
    _fields_ = [("lr", C.c_double), ("weight_decay", C.c_double), ("beta2", C.c_double), ("eps", C.c_double),
                ("eps_floor", C.c_double), ("root_tol", C.c_double), ("step", C.c_int64), ("root_every", C.c_int32),
                ("max_root_iters", C.c_int32), ("flags", C.c_uint32), ("reserved", C.c_uint32)]

    def __init__(self, lr=1e-3, weight_decay=0.0, beta2=1.0, eps=1e-6, eps_floor=2.0 ** -20, root_tol=0.0, step=1,
                 root_every=1, max_root_iters=0, flags=0):
        super().__init__(lr, weight_decay, beta2, eps, eps_floor, root_tol, step, root_every, max_root_iters, flags, 0)


class Caps(C.Structure):             # mfsdp_caps_t
    _fields_ = [("owner_num", C.c_uint32), ("owner_den", C.c_uint32), ("ws_num", C.c_uint32), ("ws_den", C.c_uint32),
                ("abs_owner_bytes", C.c_uint64), ("abs_ws_bytes", C.c_uint64)]

    def __init__(self, owner_num=9, owner_den=8, ws_num=9, ws_den=8, abs_owner_bytes=0, abs_ws_bytes=0):
        super().__init__(owner_num, owner_den, ws_num, ws_den, abs_owner_bytes, abs_ws_bytes)


class RankScore(C.Structure):        # mfsdp_rank_score_t
    _fields_ = [(n, C.c_uint64) for n in ("param_bytes", "grad_bytes", "state_bytes", "comm_bytes", "workspace_bytes",
                                          "max_block_owner_bytes")]


class BlockScore(C.Structure):       # mfsdp_block_score_t
    _fields_ = [("block_id", C.c_uint32), ("reserved", C.c_uint32), ("param_bytes", C.c_uint64),
                ("max_owner_bytes", C.c_uint64), ("gamma", C.c_double), ("c_fsdp", C.c_double), ("c_owner", C.c_double)]


class ReduceOp(C.Structure):         # mfsdp_reduce_op_t
    _fields_ = [("seq", C.c_uint32), ("role", C.c_uint32), ("kind", C.c_uint32), ("block_id", C.c_uint32),
                ("param_id", C.c_uint32), ("owner", C.c_uint32), ("dtype", C.c_uint32), ("flag", C.c_int32),
                ("numel", C.c_uint64), ("owner_elem_off", C.c_uint64)]


class MfsdpError(RuntimeError):
    def __init__(self, code, what):
        self.code = code
        super().__init__("%s failed: %d (%s)" % (what, code, mfsdp_strerror(code)))


@dataclass
class PlanResult:
    owner: list          # owner rank per role, roles in model order
    n_roles: int
    rank_load: list      # [2 * world]: primary loads then tail loads
    desc: object         # ctypes array of Desc (the chosen rank's resident set)
    rank: int
    policy_used: int = -1


_SYMBOLS = ["mfsdp_plan", "mfsdp_plan_ex", "mfsdp_score_plan", "mfsdp_reduce_schedule", "mfsdp_muon_step_gated", "mfsdp_muon_step_fanout",
            "mfsdp_signal_ready", "mfsdp_validate_desc", "mfsdp_flat_elems", "mfsdp_workspace_bytes",
            "mfsdp_workspace_view", "mfsdp_muon_step", "mfsdp_muon_momentum_pass", "mfsdp_muon_ns_pass",
            "mfsdp_muon_update_pass", "mfsdp_muon_step_host", "mfsdp_host_workspace_bytes", "mfsdp_adamw_tail_step", "mfsdp_debug_ws_offsets",
            "mfsdp_strerror", "mfsdp_version", "mfsdp_launch_count", "mfsdp_tune", "mfsdp_get_tune", "mfsdp_debug_trace",
            "mfsdp_release_plans", "mfsdp_ns_class", "mfsdp_shampoo_state_bytes", "mfsdp_shampoo_workspace_bytes",
            "mfsdp_shampoo_step", "mfsdp_shampoo_view", "mfsdp_momentum_pass_static", "mfsdp_static_max_elems"]
_lib = None


def lib_path():
    return os.path.join(PKG, "libmfsdp.so")


def exported_symbols():
    return list(_SYMBOLS)


def load():
    """dlopen libmfsdp.so (built in-tree by paper_2607_05895_b200.build).  Raises if it is missing: no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise RuntimeError("libmfsdp.so is not built (%s); run `python -m paper_2607_05895_b200.build` -- there is "
                           "no CPU fallback" % path)
    lib = C.CDLL(path)
    vp, sz, i32 = C.c_void_p, C.c_size_t, C.c_int
    pD, pP = C.POINTER(Desc), C.POINTER(Param)
    psz = C.POINTER(C.c_size_t)
    lib.mfsdp_plan.argtypes = [pP, sz, i32, i32, i32, i32, C.POINTER(C.c_int32), psz, C.POINTER(C.c_uint64), pD, sz,
                               psz, C.POINTER(C.c_int)]
    lib.mfsdp_plan_ex.argtypes = [pP, sz, i32, i32, i32, i32, C.POINTER(Caps), C.POINTER(C.c_int32), psz,
                                  C.POINTER(C.c_uint64), pD, sz, psz, C.POINTER(C.c_int), C.POINTER(C.c_int)]
    lib.mfsdp_score_plan.argtypes = [pP, sz, i32, C.POINTER(C.c_int32), sz, C.POINTER(RankScore), C.POINTER(BlockScore),
                                     sz, psz]
    lib.mfsdp_reduce_schedule.argtypes = [pP, sz, i32, C.POINTER(C.c_int32), sz, i32, C.POINTER(ReduceOp), sz, psz,
                                          C.POINTER(C.c_uint64)]
    lib.mfsdp_validate_desc.argtypes = [pD, sz]
    lib.mfsdp_flat_elems.argtypes = [pD, sz, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
    lib.mfsdp_workspace_bytes.argtypes = [pD, sz, i32, psz]
    lib.mfsdp_host_workspace_bytes.argtypes = [pD, sz, i32, psz]
    lib.mfsdp_workspace_view.argtypes = [pD, sz, i32, i32, sz, psz, psz, psz]
    lib.mfsdp_debug_ws_offsets.argtypes = [pD, sz, i32, sz, psz]
    pMH, pAH = C.POINTER(MuonHParams), C.POINTER(AdamWHParams)
    lib.mfsdp_muon_step.argtypes = [pD, sz, vp, vp, vp, vp, sz, pMH, vp]
    lib.mfsdp_muon_step_gated.argtypes = [pD, sz, vp, vp, vp, vp, sz, pMH, vp, C.c_uint32, vp]
    lib.mfsdp_signal_ready.argtypes = [vp, sz, C.c_uint32, vp]
    lib.mfsdp_muon_step_fanout.argtypes = [pD, sz, vp, vp, vp, vp, sz, pMH, C.POINTER(C.c_void_p), vp]
    lib.mfsdp_muon_momentum_pass.argtypes = [pD, sz, vp, vp, vp, sz, pMH, vp]
    lib.mfsdp_muon_ns_pass.argtypes = [pD, sz, vp, sz, pMH, vp]
    lib.mfsdp_muon_update_pass.argtypes = [pD, sz, vp, vp, sz, pMH, vp]
    lib.mfsdp_muon_step_host.argtypes = [pD, sz, vp, vp, vp, vp, vp, vp, i32, vp, sz, pMH, vp]
    lib.mfsdp_adamw_tail_step.argtypes = [pD, sz, vp, vp, vp, vp, pAH, vp]
    lib.mfsdp_momentum_pass_static.argtypes = [C.c_uint32, C.c_uint32, i32, i32, vp, vp, vp, vp, vp, pMH, vp]
    lib.mfsdp_static_max_elems.restype = C.c_uint64
    lib.mfsdp_strerror.argtypes = [i32]
    lib.mfsdp_strerror.restype = C.c_char_p
    lib.mfsdp_version.restype = i32
    lib.mfsdp_launch_count.restype = C.c_uint64
    lib.mfsdp_tune.argtypes = [i32, i32]
    lib.mfsdp_get_tune.argtypes = [i32]
    lib.mfsdp_debug_trace.argtypes = [vp, sz]
    lib.mfsdp_ns_class.argtypes = [C.c_uint32, C.c_uint32]
    lib.mfsdp_shampoo_state_bytes.argtypes = [pD, sz, psz]
    lib.mfsdp_shampoo_workspace_bytes.argtypes = [pD, sz, C.c_uint32, psz, psz]
    lib.mfsdp_shampoo_view.argtypes = [pD, sz, C.c_uint32, sz, psz]
    lib.mfsdp_shampoo_step.argtypes = [pD, sz, vp, vp, vp, sz, vp, sz, C.POINTER(ShampooHParams), vp]
    for name in _SYMBOLS:
        getattr(lib, name)          # AttributeError if the library does not export what the header declares
    _lib = lib
    return lib


# ---- marshalling helpers ----------------------------------------------------------------------------------------
def _ptr(x):
    """Device/host pointer of a torch tensor, an int address, or None."""
    if x is None:
        return None
    if isinstance(x, int):
        return C.c_void_p(x)
    return C.c_void_p(x.data_ptr())


def _nbytes(x):
    return x.numel() * x.element_size()


def _stream(stream):
    if stream is None:
        import torch
        if torch.cuda.is_available():
            return C.c_void_p(torch.cuda.current_stream().cuda_stream)
        return None
    if isinstance(stream, int):
        return C.c_void_p(stream)
    return C.c_void_p(stream.cuda_stream)


def make_desc_array(desc):
    """ctypes Desc array from a Desc array (returned as is), a list of Desc, or a list of dicts."""
    if isinstance(desc, C.Array):
        return desc
    arr = (Desc * max(1, len(desc)))()
    for i, d in enumerate(desc):
        if isinstance(d, Desc):
            arr[i] = d
        else:
            arr[i] = Desc(d["role"], d["param_id"], d["block_id"], d["rows"], d["cols"], d["dtype"], d["flags"], 0,
                          d["elem_off"])
    arr._n = len(desc)
    return arr


def _dn(desc):
    arr = make_desc_array(desc)
    return arr, getattr(arr, "_n", len(arr))


def _check(rc, what):
    if rc != 0:
        raise MfsdpError(rc, what)


# ---- the C ABI, same names ----------------------------------------------------------------------------------------
def mfsdp_strerror(code):
    return load().mfsdp_strerror(code).decode()


def mfsdp_version():
    return load().mfsdp_version()


def mfsdp_launch_count():
    return int(load().mfsdp_launch_count())


TUNE_PAIR_MIN_D, TUNE_SYM_BAND, TUNE_SYM_BAND2, TUNE_RECT_GROUP, TUNE_WIDE_MIN_KB, TUNE_FUSED_BELOW_D, TUNE_FUSED2_BELOW_D = 0, 1, 2, 3, 4, 5, 6


def mfsdp_ns_class(rows, cols):
    v = load().mfsdp_ns_class(int(rows), int(cols))
    if v < 0:
        _check(v, "mfsdp_ns_class")
    return v


def mfsdp_release_plans():
    _check(load().mfsdp_release_plans(), "mfsdp_release_plans")


def mfsdp_tune(knob, value):
    _check(load().mfsdp_tune(int(knob), int(value)), "mfsdp_tune")


def mfsdp_debug_trace(buf):
    """buf: zeroed int64 CUDA tensor (kept alive by the caller) or None to switch tracing off."""
    if buf is None:
        _check(load().mfsdp_debug_trace(None, 0), "mfsdp_debug_trace")
    else:
        _check(load().mfsdp_debug_trace(_ptr(buf), buf.numel() * buf.element_size()), "mfsdp_debug_trace")


def mfsdp_get_tune(knob):
    v = load().mfsdp_get_tune(int(knob))
    if v < 0:
        _check(v, "mfsdp_get_tune")
    return v


def _param_array(params):
    n = len(params)
    arr = (Param * max(1, n))()
    for i, p in enumerate(params):
        arr[i] = p if isinstance(p, Param) else Param(*p)
    return arr, n


def mfsdp_plan_ex(params, world_size, policy=POLICY_ROLE_GREEDY, metric=METRIC_NUMEL, rank=0, caps=None):
    """params: list of (block_id, ndim, rows, cols, dtype, flags) tuples or Param; caps: Caps or None (defaults).
    Returns PlanResult (policy_used = ROLE_GREEDY / SCOPE_GREEDY actually taken)."""
    lib = load()
    arr, n = _param_array(params)
    cp = C.byref(caps) if caps is not None else None
    n_roles, n_desc, rank_out, used = C.c_size_t(0), C.c_size_t(0), C.c_int(0), C.c_int(0)
    rc = lib.mfsdp_plan_ex(arr, n, world_size, policy, metric, rank, cp, None, C.byref(n_roles), None, None, 0,
                           C.byref(n_desc), C.byref(rank_out), C.byref(used))
    _check(rc, "mfsdp_plan_ex(size query)")
    owner = (C.c_int32 * max(1, n_roles.value))()
    loads = (C.c_uint64 * (2 * world_size))()
    desc = (Desc * max(1, n_desc.value))()
    cap = n_desc.value
    rc = lib.mfsdp_plan_ex(arr, n, world_size, policy, metric, rank, cp, owner, C.byref(n_roles), loads, desc, cap,
                           C.byref(n_desc), C.byref(rank_out), C.byref(used))
    _check(rc, "mfsdp_plan_ex")
    desc._n = n_desc.value
    return PlanResult(list(owner[:n_roles.value]), n_roles.value, list(loads), desc, rank_out.value, used.value)


def mfsdp_plan(params, world_size, policy=POLICY_ROLE_GREEDY, metric=METRIC_NUMEL, rank=0):
    """params: list of (block_id, ndim, rows, cols, dtype, flags) tuples or Param.  Returns PlanResult."""
    lib = load()
    arr, n = _param_array(params)
    n_roles, n_desc, rank_out = C.c_size_t(0), C.c_size_t(0), C.c_int(0)
    rc = lib.mfsdp_plan(arr, n, world_size, policy, metric, rank, None, C.byref(n_roles), None, None, 0,
                        C.byref(n_desc), C.byref(rank_out))
    _check(rc, "mfsdp_plan(size query)")
    owner = (C.c_int32 * max(1, n_roles.value))()
    loads = (C.c_uint64 * (2 * world_size))()
    desc = (Desc * max(1, n_desc.value))()
    cap = n_desc.value
    rc = lib.mfsdp_plan(arr, n, world_size, policy, metric, rank, owner, C.byref(n_roles), loads, desc, cap,
                        C.byref(n_desc), C.byref(rank_out))
    _check(rc, "mfsdp_plan")
    desc._n = n_desc.value
    return PlanResult(list(owner[:n_roles.value]), n_roles.value, list(loads), desc, rank_out.value)


def mfsdp_score_plan(params, world_size, owner):
    """(list of RankScore per rank, list of BlockScore per block in model order) of a completed plan."""
    lib = load()
    arr, n = _param_array(params)
    own = (C.c_int32 * max(1, len(owner)))(*owner)
    nb = C.c_size_t(0)
    _check(lib.mfsdp_score_plan(arr, n, world_size, own, len(owner), None, None, 0, C.byref(nb)), "mfsdp_score_plan(size)")
    ranks = (RankScore * world_size)()
    blocks = (BlockScore * max(1, nb.value))()
    _check(lib.mfsdp_score_plan(arr, n, world_size, own, len(owner), ranks, blocks, nb.value, C.byref(nb)),
           "mfsdp_score_plan")
    return list(ranks), list(blocks[:nb.value])


def mfsdp_validate_desc(desc):
    arr, n = _dn(desc)
    return load().mfsdp_validate_desc(arr, n)


def mfsdp_flat_elems(desc):
    arr, n = _dn(desc)
    a, b = C.c_uint64(0), C.c_uint64(0)
    _check(load().mfsdp_flat_elems(arr, n, C.byref(a), C.byref(b)), "mfsdp_flat_elems")
    return a.value, b.value


def mfsdp_workspace_bytes(desc, precision=NS_BF16):
    arr, n = _dn(desc)
    out = C.c_size_t(0)
    _check(load().mfsdp_workspace_bytes(arr, n, precision, C.byref(out)), "mfsdp_workspace_bytes")
    return out.value


def mfsdp_host_workspace_bytes(desc, precision=NS_BF16):
    arr, n = _dn(desc)
    out = C.c_size_t(0)
    _check(load().mfsdp_host_workspace_bytes(arr, n, precision, C.byref(out)), "mfsdp_host_workspace_bytes")
    return out.value


def mfsdp_workspace_view(desc, precision, ns_steps, index):
    """(o_byte_off, o_pitch_elems, ssq_byte_off) of the index-th matrix descriptor."""
    arr, n = _dn(desc)
    a, b, c = C.c_size_t(0), C.c_size_t(0), C.c_size_t(0)
    _check(load().mfsdp_workspace_view(arr, n, precision, ns_steps, index, C.byref(a), C.byref(b), C.byref(c)),
           "mfsdp_workspace_view")
    return a.value, b.value, c.value


def mfsdp_debug_ws_offsets(desc, precision, index):
    arr, n = _dn(desc)
    out = (C.c_size_t * 6)()
    _check(load().mfsdp_debug_ws_offsets(arr, n, precision, index, out), "mfsdp_debug_ws_offsets")
    return list(out)


def mfsdp_muon_step(desc, W, G, M, workspace, hp, stream=None):
    arr, n = _dn(desc)
    _check(load().mfsdp_muon_step(arr, n, _ptr(W), _ptr(G), _ptr(M), _ptr(workspace), _nbytes(workspace),
                                  C.byref(hp), _stream(stream)), "mfsdp_muon_step")


def mfsdp_muon_step_gated(desc, W, G, M, workspace, hp, ready, epoch, stream=None):
    """ready: uint32/int32 CUDA tensor, one flag per matrix descriptor; the momentum pass of matrix i waits for
    ready[i] >= epoch."""
    arr, n = _dn(desc)
    _check(load().mfsdp_muon_step_gated(arr, n, _ptr(W), _ptr(G), _ptr(M), _ptr(workspace), _nbytes(workspace),
                                        C.byref(hp), _ptr(ready), int(epoch), _stream(stream)), "mfsdp_muon_step_gated")


def mfsdp_muon_step_fanout(desc, W, G, M, workspace, hp, fanout, stream=None):
    """fanout: one entry per matrix descriptor -- a CUDA tensor (or int address) that receives the updated matrix, or
    None."""
    arr, n = _dn(desc)
    ptrs = (C.c_void_p * max(1, len(fanout)))(*[None if t is None else (t if isinstance(t, int) else t.data_ptr())
                                                for t in fanout])
    _check(load().mfsdp_muon_step_fanout(arr, n, _ptr(W), _ptr(G), _ptr(M), _ptr(workspace), _nbytes(workspace),
                                         C.byref(hp), ptrs, _stream(stream)), "mfsdp_muon_step_fanout")


def mfsdp_signal_ready(ready, index, epoch, stream=None):
    _check(load().mfsdp_signal_ready(_ptr(ready), int(index), int(epoch), _stream(stream)), "mfsdp_signal_ready")


def mfsdp_reduce_schedule(params, world_size, owner, reverse_blocks=True):
    """(list of ReduceOp, 64-bit validation hash) of the owner-segment gradient reduction."""
    lib = load()
    arr, n = _param_array(params)
    own = (C.c_int32 * max(1, len(owner)))(*owner)
    n_ops, h = C.c_size_t(0), C.c_uint64(0)
    _check(lib.mfsdp_reduce_schedule(arr, n, world_size, own, len(owner), int(reverse_blocks), None, 0, C.byref(n_ops),
                                     C.byref(h)), "mfsdp_reduce_schedule(size)")
    ops = (ReduceOp * max(1, n_ops.value))()
    _check(lib.mfsdp_reduce_schedule(arr, n, world_size, own, len(owner), int(reverse_blocks), ops, n_ops.value,
                                     C.byref(n_ops), C.byref(h)), "mfsdp_reduce_schedule")
    return list(ops[:n_ops.value]), h.value


def mfsdp_muon_momentum_pass(desc, G, M, workspace, hp, stream=None):
    arr, n = _dn(desc)
    _check(load().mfsdp_muon_momentum_pass(arr, n, _ptr(G), _ptr(M), _ptr(workspace), _nbytes(workspace),
                                           C.byref(hp), _stream(stream)), "mfsdp_muon_momentum_pass")


def mfsdp_static_max_elems():
    """Largest rows * cols mfsdp_momentum_pass_static accepts (the size of its built-in scratch array)."""
    return int(load().mfsdp_static_max_elems())


def mfsdp_momentum_pass_static(rows, cols, dtype, precision, G, M, X, ssq, inv_norm, hp, stream=None):
    """Momentum pass of one contiguous rows x cols matrix that allocates nothing on the device: for callers that cannot
    call cudaMalloc (a framework allocator owns the GPU, or the device-wide synchronisation of an allocation is not
    acceptable inside the step loop).  G: gradient (dtype), M: float momentum (in place), X: cast(U) out (bf16 for
    NS_BF16, float for NS_FP32), ssq: one float64, inv_norm: one float32 -- all CUDA tensors or addresses the caller
    owns.  Shares a fixed 512 KiB scratch array per GPU with every other call: do not let two calls overlap on one
    GPU.  Raises MfsdpError(ETOOBIG) beyond mfsdp_static_max_elems() elements.  See include/mfsdp.h."""
    _check(load().mfsdp_momentum_pass_static(int(rows), int(cols), int(dtype), int(precision), _ptr(G), _ptr(M),
                                             _ptr(X), _ptr(ssq), _ptr(inv_norm), C.byref(hp), _stream(stream)),
           "mfsdp_momentum_pass_static")


def mfsdp_muon_ns_pass(desc, workspace, hp, stream=None):
    arr, n = _dn(desc)
    _check(load().mfsdp_muon_ns_pass(arr, n, _ptr(workspace), _nbytes(workspace), C.byref(hp), _stream(stream)),
           "mfsdp_muon_ns_pass")


def mfsdp_muon_update_pass(desc, W, workspace, hp, stream=None):
    arr, n = _dn(desc)
    _check(load().mfsdp_muon_update_pass(arr, n, _ptr(W), _ptr(workspace), _nbytes(workspace), C.byref(hp),
                                         _stream(stream)), "mfsdp_muon_update_pass")


def mfsdp_muon_step_host(desc, hW, hG, hM, dW, dG, dM, upload_state, workspace, hp, stream=None):
    """HOST buffers hW/hG/hM (pinned torch CPU tensors), device staging dW/dG/dM.  Synchronises the stream."""
    arr, n = _dn(desc)
    _check(load().mfsdp_muon_step_host(arr, n, _ptr(hW), _ptr(hG), _ptr(hM), _ptr(dW), _ptr(dG), _ptr(dM),
                                       int(upload_state), _ptr(workspace), _nbytes(workspace), C.byref(hp),
                                       _stream(stream)), "mfsdp_muon_step_host")


def mfsdp_adamw_tail_step(desc, P, G, m, v, hp, stream=None):
    arr, n = _dn(desc)
    _check(load().mfsdp_adamw_tail_step(arr, n, _ptr(P), _ptr(G), _ptr(m), _ptr(v), C.byref(hp), _stream(stream)),
           "mfsdp_adamw_tail_step")


def mfsdp_shampoo_state_bytes(desc):
    arr, n = _dn(desc)
    out = C.c_size_t(0)
    _check(load().mfsdp_shampoo_state_bytes(arr, n, C.byref(out)), "mfsdp_shampoo_state_bytes")
    return out.value


def mfsdp_shampoo_workspace_bytes(desc, flags=0):
    """(min_bytes, full_bytes)"""
    arr, n = _dn(desc)
    lo, hi = C.c_size_t(0), C.c_size_t(0)
    _check(load().mfsdp_shampoo_workspace_bytes(arr, n, flags, C.byref(lo), C.byref(hi)), "mfsdp_shampoo_workspace_bytes")
    return lo.value, hi.value


def mfsdp_shampoo_view(desc, flags, index):
    arr, n = _dn(desc)
    out = (C.c_size_t * 12)()
    _check(load().mfsdp_shampoo_view(arr, n, flags, index, out), "mfsdp_shampoo_view")
    return list(out)


def mfsdp_shampoo_step(desc, W, G, state, workspace, hp, stream=None):
    arr, n = _dn(desc)
    _check(load().mfsdp_shampoo_step(arr, n, _ptr(W), _ptr(G), _ptr(state), _nbytes(state), _ptr(workspace),
                                     _nbytes(workspace), C.byref(hp), _stream(stream)), "mfsdp_shampoo_step")
