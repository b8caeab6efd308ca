"""Thin ctypes binding over libfmx.so (include/fmx.h).  Argument marshalling only: every step of
the forward runs in the library's CUDA kernels.  Device buffers are passed as integer addresses
(e.g. torch.Tensor.data_ptr()); PyTorch is used by callers only for device memory and streams.

Importing this module never compiles anything; `load()` fails loudly if libfmx.so is missing
(build it with `python -m paper_2606_09643_b200.build` or `__graft_entry__.build()`).
"""
import ctypes as C
import math
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfmx.so")

FMX_OK = 0
STATUS = {0: "FMX_OK", -1: "FMX_E_INVALID_ARG", -2: "FMX_E_UNKNOWN_BACKBONE", -3: "FMX_E_UNKNOWN_TASK",
          -4: "FMX_E_SHAPE", -5: "FMX_E_BAD_LENGTH", -6: "FMX_E_WORKSPACE", -7: "FMX_E_CAPACITY", -8: "FMX_E_CUDA"}
ACT = {"gelu": 0, "relu": 1, "swiglu": 2}
NORM = {"ln": 0, "rms": 1}
INPUT_KIND = {"embedded": 0, "patch": 1, "tokens": 2}
TARGET = {"q": 0, "k": 1, "v": 2, "o": 3, "gate": 4, "up": 5, "down": 6}
HEAD_KIND = {"mean": 0, "cls": 1, "last": 2, "flatten": 3, "dense": 4}
N_FAMILIES = 12
MAX_TASKS = 1024

_vp, _vpp = C.c_void_p, C.POINTER(C.c_void_p)


class BackboneDesc(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("n_layers", "d_model", "n_q_heads", "n_kv_heads", "head_dim", "d_ffn", "act", "norm")] + \
               [("norm_eps", C.c_float), ("causal", C.c_int32), ("rope_theta", C.c_float)] + \
               [(n, C.c_int32) for n in ("input_kind", "patch_dim", "tokens_per_request", "has_cls", "vocab", "max_seq",
                                         "img_c", "img_hw", "patch_hw")] + \
               [(n, _vp) for n in ("embed_W", "embed_b", "embed_cls", "embed_pos", "embed_table")] + \
               [(n, _vpp) for n in ("norm1_g", "norm1_b", "Wq", "Wk", "Wv", "Wo", "bq", "bk", "bv", "bo", "norm2_g", "norm2_b",
                                    "Wup", "Wgate", "Wdown", "bup", "bgate", "bdown")] + \
               [("final_g", _vp), ("final_b", _vp), ("rel_bias", _vp), ("rel_buckets", C.c_int32), ("rel_max_distance", C.c_int32)]


class AdapterDesc(C.Structure):
    _fields_ = [("target", C.c_int32), ("rank", C.c_int32), ("scaling", C.c_float), ("A", _vpp), ("B", _vpp)]


class TaskDesc(C.Structure):
    _fields_ = [("n_adapters", C.c_int32), ("adapters", C.POINTER(AdapterDesc)), ("head_kind", C.c_int32),
                ("head_out", C.c_int32), ("head_W", _vp), ("head_b", _vp),
                ("head_hidden", C.c_int32), ("head_W2", _vp), ("head_b2", _vp),
                ("enc_channels", C.c_int32), ("enc_W", _vp), ("enc_b", _vp)]


class BfqParams(C.Structure):
    _fields_ = [("n_tasks", C.c_int32), ("b_max", C.c_int32), ("lat_ms", C.POINTER(C.c_double)), ("l_tok_ms", C.c_double)]


OPTIONS = {"attention_impl": 0, "pdl": 2, "shrink_stages": 3, "half_tiles": 4, "attn_short": 5, "rope_fused": 6, "head_tiled": 7, "shrink_fused": 8, "graph": 9, "reverse": 10, "expand_wide": 11, "deep_pipe": 12, "decode_fork": 13, "decode_rowgemm": 14, "embed_small": 15}


class FmxError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{STATUS.get(code, code)}: {msg}")
        self.code = code


_lib = None

# include/fmx.h (the public C ABI)
EXPORTS = ["fmx_create", "fmx_destroy", "fmx_last_error", "fmx_version", "fmx_poll_error", "fmx_register_backbone", "fmx_register_task",
           "fmx_unregister_task", "fmx_output_layout", "fmx_output_layout_len", "fmx_workspace_bytes", "fmx_host_workspace_bytes", "fmx_forward_mixed",
           "fmx_forward_mixed_host", "fmx_register_lm_head", "fmx_kv_cache_bytes", "fmx_prefill", "fmx_decode_step", "fmx_row_gemm_static", "fmx_debug_get_segments", "fmx_task_slots", "fmx_profile_enable", "fmx_profile_select",
           "fmx_profile_read", "fmx_profile_family_name", "fmx_last_launch_count", "fmx_bfq_create", "fmx_bfq_destroy",
           "fmx_bfq_set_task", "fmx_bfq_enqueue", "fmx_bfq_next_batch", "fmx_bfq_complete", "fmx_bfq_stats", "fmx_bfq_peek"]
# csrc/fmx_internal.h (test hooks and tuning knobs; not part of the ABI)
INTERNAL_EXPORTS = ["fmx_debug_get_tiles", "fmx_debug_read", "fmx_graph_replays", "fmx_debug_gemm", "fmx_debug_attention", "fmx_set_option"]


def load():
    """dlopen libfmx.so; raises if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_09643_b200.build`; "
                                "this package has no CPU or PyTorch fallback")
    lib = C.CDLL(LIB_PATH)
    i32p, i64p, f64p = C.POINTER(C.c_int32), C.POINTER(C.c_int64), C.POINTER(C.c_double)
    lib.fmx_last_error.restype = C.c_char_p
    lib.fmx_version.restype = C.c_char_p
    lib.fmx_profile_family_name.restype = C.c_char_p
    lib.fmx_profile_family_name.argtypes = [C.c_int]
    lib.fmx_create.argtypes = [C.POINTER(_vp), C.c_int]
    lib.fmx_destroy.argtypes = [_vp]
    lib.fmx_register_backbone.argtypes = [_vp, C.POINTER(BackboneDesc), i32p]
    lib.fmx_register_task.argtypes = [_vp, C.c_int32, C.POINTER(TaskDesc), i32p]
    lib.fmx_unregister_task.argtypes = [_vp, C.c_int32]
    lib.fmx_output_layout.argtypes = [_vp, i32p, C.c_int32, i64p]
    lib.fmx_output_layout_len.argtypes = [_vp, i32p, i32p, C.c_int32, i64p]
    lib.fmx_workspace_bytes.argtypes = [_vp, C.c_int32, C.c_int32, C.c_int64, C.POINTER(C.c_size_t)]
    lib.fmx_host_workspace_bytes.argtypes = [_vp, C.c_int32, C.c_int32, C.c_int64, C.c_size_t, C.c_int64, C.POINTER(C.c_size_t)]
    lib.fmx_poll_error.argtypes = [_vp]
    lib.fmx_forward_mixed.argtypes = [_vp, C.c_int32, _vp, i32p, i32p, C.c_int32, _vp, _vp, C.c_size_t, _vp]
    lib.fmx_forward_mixed_host.argtypes = [_vp, C.c_int32, _vp, C.c_size_t, i32p, i32p, C.c_int32, _vp, _vp, C.c_size_t, _vp]
    lib.fmx_register_lm_head.argtypes = [_vp, C.c_int32, _vp, C.c_int32]
    lib.fmx_kv_cache_bytes.argtypes = [_vp, C.c_int32, C.c_int32, C.POINTER(C.c_size_t)]
    lib.fmx_prefill.argtypes = [_vp, C.c_int32, _vp, i32p, i32p, i32p, C.c_int32, _vp, _vp, _vp, _vp, C.c_int32, _vp, C.c_size_t, _vp]
    lib.fmx_decode_step.argtypes = [_vp, C.c_int32, _vp, i32p, i32p, i32p, C.c_int32, _vp, _vp, _vp, C.c_int32, _vp, C.c_size_t, _vp]
    lib.fmx_debug_get_segments.argtypes = [_vp, i32p, i32p, i32p, i32p, i32p]
    lib.fmx_debug_get_tiles.argtypes = [_vp, i32p, i32p, i32p, C.c_int32]
    lib.fmx_task_slots.argtypes = [_vp]
    lib.fmx_debug_read.argtypes = [_vp, C.c_int, _vp, C.c_size_t]
    lib.fmx_profile_enable.argtypes = [_vp, C.c_int]
    lib.fmx_profile_select.argtypes = [_vp, C.c_uint32]
    lib.fmx_profile_read.argtypes = [_vp, i32p, f64p]
    lib.fmx_last_launch_count.argtypes = [_vp]
    lib.fmx_graph_replays.argtypes = [_vp]
    lib.fmx_graph_replays.restype = C.c_longlong
    lib.fmx_debug_gemm.argtypes = [_vp, _vp, _vp, _vp, C.c_int32, C.c_int32, C.c_int32, _vp]
    lib.fmx_row_gemm_static.argtypes = [_vp, _vp, _vp, C.c_int32, C.c_int32, C.c_int32, _vp]
    lib.fmx_debug_attention.argtypes = [_vp, _vp, _vp, i32p, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, _vp]
    lib.fmx_set_option.argtypes = [_vp, C.c_int32, C.c_int32]
    lib.fmx_bfq_create.argtypes = [C.POINTER(BfqParams), C.POINTER(_vp)]
    lib.fmx_bfq_destroy.argtypes = [_vp]
    lib.fmx_bfq_set_task.argtypes = [_vp, C.c_int32, C.c_double, C.c_double]
    lib.fmx_bfq_enqueue.argtypes = [_vp, C.c_int32, C.c_uint64, C.c_int32, C.c_double]
    lib.fmx_bfq_next_batch.argtypes = [_vp, C.c_double, C.c_int32, i32p, i32p, C.POINTER(C.c_uint64), i32p]
    lib.fmx_bfq_complete.argtypes = [_vp, C.c_double]
    lib.fmx_bfq_stats.argtypes = [_vp, C.c_int32, i64p, f64p, i32p]
    lib.fmx_bfq_peek.argtypes = [_vp, C.c_int32, C.c_int32, f64p]
    _lib = lib
    return lib


def _check(code):
    if code != FMX_OK:
        raise FmxError(code, load().fmx_last_error().decode())


def row_gemm_static(x, W, out, M, N, K, stream=0):
    """fmx_row_gemm_static: out[M, N] fp32 = x[M, K] . W[N, K]^T (bf16 device pointers) on the current device; allocates nothing
    (its scratch is a static 8 MiB device array), M <= 128.  Calls that overlap on the GPU race on that array."""
    _check(load().fmx_row_gemm_static(x, W, out, M, N, K, stream or None))


def _ptr_array(ptrs):
    """list of device addresses (or None) -> ctypes array of void*; None list -> NULL."""
    if ptrs is None:
        return None
    arr = (C.c_void_p * len(ptrs))(*[C.c_void_p(p) if p else None for p in ptrs])
    return arr


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


class Fmx:
    """One fmx_ctx.  Methods mirror the C entry points one to one."""

    def __init__(self, device=0):
        self.lib = load()
        self.h = _vp()
        _check(self.lib.fmx_create(C.byref(self.h), device))
        self._keep = []          # ctypes arrays that must outlive the calls that reference them

    def destroy(self):
        if self.h:
            self.lib.fmx_destroy(self.h)
            self.h = _vp()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def register_backbone(self, fields, per_layer, singles):
        """fields: dict of scalar descriptor fields; per_layer: dict name -> list of device
        addresses (len n_layers) or None; singles: dict name -> device address or None."""
        d = BackboneDesc()
        for k, v in fields.items():
            setattr(d, k, v)
        keep = []
        for k, v in per_layer.items():
            arr = _ptr_array(v)
            keep.append(arr)
            setattr(d, k, C.cast(arr, _vpp) if arr is not None else None)
        for k, v in singles.items():
            setattr(d, k, v)
        out = C.c_int32(-1)
        _check(self.lib.fmx_register_backbone(self.h, C.byref(d), C.byref(out)))
        return out.value

    def register_task(self, bb, adapters, head_kind, head_out, head_W, head_b, head_hidden=0, head_W2=None, head_b2=None,
                      enc_channels=0, enc_W=None, enc_b=None):
        """adapters: list of (target:int, rank:int, scaling:float, A_ptrs:list, B_ptrs:list).  head_hidden > 0: MLP head
        (head_W [hidden, d_feat], head_b [hidden], head_W2 [head_out, hidden], head_b2 [head_out]).  enc_channels > 1: input channel combiner (enc_W [C], enc_b [1])."""
        n = len(adapters)
        arr = (AdapterDesc * max(n, 1))()
        keep = []
        for i, (tg, rank, scaling, A, B) in enumerate(adapters):
            a, b = _ptr_array(A), _ptr_array(B)
            keep += [a, b]
            arr[i].target, arr[i].rank, arr[i].scaling = tg, rank, scaling
            arr[i].A, arr[i].B = C.cast(a, _vpp), C.cast(b, _vpp)
        d = TaskDesc(n, arr if n else None, head_kind, head_out, head_W, head_b, head_hidden, head_W2, head_b2, enc_channels, enc_W, enc_b)
        out = C.c_int32(-1)
        _check(self.lib.fmx_register_task(self.h, bb, C.byref(d), C.byref(out)))
        return out.value

    def unregister_task(self, task):
        _check(self.lib.fmx_unregister_task(self.h, task))

    def task_slots(self):
        return self.lib.fmx_task_slots(self.h)

    def output_layout(self, task_ids, lengths=None):
        """lengths: needed when a task with a dense (per-token) head runs on a variable-length backbone."""
        ids = _i32(task_ids)
        off = np.zeros(len(ids) + 1, dtype=np.int64)
        p = C.POINTER(C.c_int32)
        if lengths is None:
            _check(self.lib.fmx_output_layout(self.h, ids.ctypes.data_as(p), len(ids), off.ctypes.data_as(C.POINTER(C.c_int64))))
        else:
            lens = _i32(lengths)
            _check(self.lib.fmx_output_layout_len(self.h, ids.ctypes.data_as(p), lens.ctypes.data_as(p), len(ids), off.ctypes.data_as(C.POINTER(C.c_int64))))
        return off

    def workspace_bytes(self, bb, max_req, max_tokens):
        out = C.c_size_t(0)
        _check(self.lib.fmx_workspace_bytes(self.h, bb, max_req, max_tokens, C.byref(out)))
        return out.value

    def host_workspace_bytes(self, bb, max_req, max_tokens, max_input_bytes, max_output_floats):
        out = C.c_size_t(0)
        _check(self.lib.fmx_host_workspace_bytes(self.h, bb, max_req, max_tokens, max_input_bytes, max_output_floats, C.byref(out)))
        return out.value

    def poll_error(self):
        _check(self.lib.fmx_poll_error(self.h))

    def forward_mixed(self, bb, inputs, task_ids, lengths, outputs, workspace, workspace_bytes, stream=0):
        ids, lens = _i32(task_ids), _i32(lengths)
        p = C.POINTER(C.c_int32)
        _check(self.lib.fmx_forward_mixed(self.h, bb, inputs, ids.ctypes.data_as(p), lens.ctypes.data_as(p), len(ids),
                                          outputs, workspace, workspace_bytes, stream or None))

    def forward_mixed_host(self, bb, inputs_host, inputs_bytes, task_ids, lengths, outputs_host, workspace,
                           workspace_bytes, stream=0):
        ids, lens = _i32(task_ids), _i32(lengths)
        p = C.POINTER(C.c_int32)
        _check(self.lib.fmx_forward_mixed_host(self.h, bb, inputs_host, inputs_bytes, ids.ctypes.data_as(p),
                                               lens.ctypes.data_as(p), len(ids), outputs_host, workspace,
                                               workspace_bytes, stream or None))

    def register_lm_head(self, bb, W, vocab):
        _check(self.lib.fmx_register_lm_head(self.h, bb, W, vocab))

    def kv_cache_bytes(self, bb, n_slots):
        out = C.c_size_t(0)
        _check(self.lib.fmx_kv_cache_bytes(self.h, bb, n_slots, C.byref(out)))
        return out.value

    def prefill(self, bb, inputs, task_ids, lengths, slots, outputs, scores, next_tokens, kv_cache, n_slots, workspace, workspace_bytes, stream=0):
        ids, lens, sl = _i32(task_ids), _i32(lengths), _i32(slots)
        p = C.POINTER(C.c_int32)
        _check(self.lib.fmx_prefill(self.h, bb, inputs, ids.ctypes.data_as(p), lens.ctypes.data_as(p), sl.ctypes.data_as(p), len(ids),
                                    outputs or None, scores or None, next_tokens or None, kv_cache, n_slots, workspace, workspace_bytes, stream or None))

    def decode_step(self, bb, tokens, task_ids, slots, positions, scores, next_tokens, kv_cache, n_slots, workspace, workspace_bytes, stream=0):
        ids, sl, pos = _i32(task_ids), _i32(slots), _i32(positions)
        p = C.POINTER(C.c_int32)
        _check(self.lib.fmx_decode_step(self.h, bb, tokens, ids.ctypes.data_as(p), sl.ctypes.data_as(p), pos.ctypes.data_as(p), len(ids),
                                        scores or None, next_tokens or None, kv_cache, n_slots, workspace, workspace_bytes, stream or None))

    def debug_get_segments(self, n_req):
        T = self.task_slots()
        out = dict(perm=np.zeros(n_req, np.int32), inv_perm=np.zeros(n_req, np.int32),
                   task_req_off=np.zeros(T + 1, np.int32), cu_tok=np.zeros(n_req + 1, np.int32),
                   task_tok_off=np.zeros(T + 1, np.int32))
        p = C.POINTER(C.c_int32)
        _check(self.lib.fmx_debug_get_segments(self.h, *[out[k].ctypes.data_as(p) for k in
                                                         ("perm", "inv_perm", "task_req_off", "cu_tok", "task_tok_off")]))
        return out

    def debug_get_tiles(self, cap=1 << 16):
        nt, nb = C.c_int32(0), C.c_int32(0)
        blocks = np.zeros(4 * cap, np.int32)
        _check(self.lib.fmx_debug_get_tiles(self.h, C.byref(nt), C.byref(nb), blocks.ctypes.data_as(C.POINTER(C.c_int32)), cap))
        return nt.value, nb.value, blocks[:4 * min(nb.value, cap)].reshape(-1, 4)

    def debug_read(self, which, shape, dtype):
        """which: 0 X f32, 1 Xn, 2 QKV, 3 attn out, 4 FFN hidden, 5 U (bf16 as uint16), 6 feat f32."""
        out = np.zeros(shape, dtype=dtype)
        _check(self.lib.fmx_debug_read(self.h, which, out.ctypes.data_as(_vp), out.nbytes))
        return out

    def profile_enable(self, on=True):
        _check(self.lib.fmx_profile_enable(self.h, 1 if on else 0))

    def profile_select(self, families=None):
        """families: iterable of family names (None = all) that get events while profiling is on."""
        names = [self.lib.fmx_profile_family_name(i).decode() for i in range(N_FAMILIES)]
        mask = 0xFFFFFFFF if families is None else sum(1 << names.index(f) for f in families)
        _check(self.lib.fmx_profile_select(self.h, mask))

    def profile_read(self):
        n = np.zeros(N_FAMILIES, np.int32)
        ms = np.zeros(N_FAMILIES, np.float64)
        _check(self.lib.fmx_profile_read(self.h, n.ctypes.data_as(C.POINTER(C.c_int32)), ms.ctypes.data_as(C.POINTER(C.c_double))))
        return {self.lib.fmx_profile_family_name(i).decode(): (int(n[i]), float(ms[i])) for i in range(N_FAMILIES)}

    def last_launch_count(self):
        return self.lib.fmx_last_launch_count(self.h)

    def graph_replays(self):
        return int(self.lib.fmx_graph_replays(self.h))

    def debug_gemm(self, A, W, Cout, M, N, K, stream=0):
        _check(self.lib.fmx_debug_gemm(self.h, A, W, Cout, M, N, K, stream or None))

    def debug_attention(self, qkv, out, cu_tok, n_q_heads, n_kv_heads, head_dim, causal, impl=0, stream=0):
        cu = np.ascontiguousarray(cu_tok, dtype=np.int32)
        _check(self.lib.fmx_debug_attention(self.h, qkv, out, cu.ctypes.data_as(C.POINTER(C.c_int32)), len(cu) - 1, n_q_heads,
                                            n_kv_heads, head_dim, int(causal), impl, stream or None))

    def set_option(self, option, value):
        """option: a key of OPTIONS (csrc/fmx_internal.h), e.g. 'attention_impl' (0 auto, 1 mma.sync, 2 tcgen05), 'pdl' (0 / 1 / 2)."""
        _check(self.lib.fmx_set_option(self.h, OPTIONS[option], int(value)))


class Bfq:
    """fmx_bfq_*: the host-side batch-aware fair-queue batch builder (no CUDA needed)."""

    def __init__(self, n_tasks, b_max, lat_ms, l_tok_ms=0.0):
        self.lib = load()
        lat = (C.c_double * b_max)(*lat_ms)
        p = BfqParams(n_tasks, b_max, lat, l_tok_ms)
        self.h = _vp()
        _check(self.lib.fmx_bfq_create(C.byref(p), C.byref(self.h)))
        self.b_max = b_max

    def __del__(self):
        try:
            if self.h:
                self.lib.fmx_bfq_destroy(self.h)
                self.h = _vp()
        except Exception:
            pass

    def set_task(self, task, weight, slo_ms=math.inf):
        _check(self.lib.fmx_bfq_set_task(self.h, task, weight, slo_ms))

    def enqueue(self, task, handle, length, arrival_ms):
        _check(self.lib.fmx_bfq_enqueue(self.h, task, handle, length, arrival_ms))

    def next_batch(self, now_ms, cap):
        n_max = max(min(self.b_max, cap), 1)
        ids, lens = np.zeros(n_max, np.int32), np.zeros(n_max, np.int32)
        handles = np.zeros(n_max, np.uint64)
        n = C.c_int32(0)
        p = C.POINTER(C.c_int32)
        _check(self.lib.fmx_bfq_next_batch(self.h, now_ms, cap, ids.ctypes.data_as(p), lens.ctypes.data_as(p),
                                           handles.ctypes.data_as(C.POINTER(C.c_uint64)), C.byref(n)))
        return ids[:n.value], lens[:n.value], handles[:n.value]

    def complete(self, measured_ms=0.0):
        _check(self.lib.fmx_bfq_complete(self.h, measured_ms))

    def stats(self, task):
        d, s, q = C.c_int64(0), C.c_double(0), C.c_int32(0)
        _check(self.lib.fmx_bfq_stats(self.h, task, C.byref(d), C.byref(s), C.byref(q)))
        return d.value, s.value, q.value

    def peek(self, task, j):
        out = (C.c_double * 3)()
        _check(self.lib.fmx_bfq_peek(self.h, task, j, out))
        return tuple(out)
