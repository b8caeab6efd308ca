"""ORACLE glue (test infrastructure): present a seeded `fmx_workloads.Workload` to the oracle.

Holds no arithmetic: it widens the workload's bf16 bit patterns to float64 and builds the
plain dicts `oracle.vfm_forward` takes.  The oracle itself never sees the workload object.
"""
from collections import OrderedDict

import numpy as np

from fmx_workloads import bf16_bits_to_f64


def bb_dict(wl):
    bb = wl.bb
    return dict(n_layers=bb.n_layers, d_model=bb.d_model, n_q_heads=bb.n_q_heads,
                n_kv_heads=bb.n_kv_heads, head_dim=bb.head_dim, d_ffn=bb.d_ffn, act=bb.act,
                norm=bb.norm, norm_eps=bb.norm_eps, causal=bb.causal, rope_theta=bb.rope_theta,
                input_kind=bb.input_kind, patch_dim=bb.patch_dim, has_cls=bb.has_cls,
                has_bias=bb.has_bias, has_pos=bb.pos_kind != "none", img_c=bb.img_c,
                img_hw=bb.img_hw, patch_hw=bb.patch_hw, rel_buckets=getattr(bb, "rel_buckets", 0),
                rel_max_distance=getattr(bb, "rel_max_distance", 0))


def task_dicts(wl):
    return [dict(id=t, adapters={a.target: (a.rank, a.scaling) for a in ts.adapters},
                 head_kind=ts.head_kind, head_out=ts.head_out, head_hidden=getattr(ts, "head_hidden", 0), enc_channels=getattr(ts, "enc_channels", 0)) for t, ts in enumerate(wl.tasks)]


def make_get(wl, max_cached_bytes=6 << 30):
    """name -> float64 array, with a byte-bounded LRU so a whole cfg4 never sits in RAM."""
    cache = OrderedDict()
    state = {"bytes": 0}

    def get(name):
        if name in cache:
            cache.move_to_end(name)
            return cache[name]
        a = bf16_bits_to_f64(wl.tensor(name))
        cache[name] = a
        state["bytes"] += a.nbytes
        while state["bytes"] > max_cached_bytes and len(cache) > 1:
            _, old = cache.popitem(last=False)
            state["bytes"] -= old.nbytes
        return a

    return get


def request_inputs(wl, indices=None):
    idx = range(wl.n_req) if indices is None else indices
    out = []
    for i in idx:
        x = wl.request_input(i)
        out.append(x if x.dtype == np.int32 else bf16_bits_to_f64(x))
    return out


def oracle_outputs(wl, indices=None):
    """Oracle outputs (list of float64 vectors) for the requests `indices` of the workload."""
    from oracle.vfm_forward import forward_requests
    idx = list(range(wl.n_req)) if indices is None else list(indices)
    return forward_requests(bb_dict(wl), make_get(wl), task_dicts(wl),
                            [int(wl.task_ids[i]) for i in idx], request_inputs(wl, idx))
