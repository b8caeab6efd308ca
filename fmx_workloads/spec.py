"""Workload specifications and seeded tensor recipes for the five BASELINE.json configs.

Everything here is *description and random draws*: shapes, distributions, seeds, task-id
draws.  No step of the vFM forward is computed here.  Each tensor has its own Philox stream
keyed by (config seed, crc32(name)), so generation is order-independent.
Values are drawn in fp32 and rounded ONCE to bf16 bit patterns (uint16); both the oracle
and the CUDA path consume exactly these bits.
"""
from __future__ import annotations

import math
import zlib
from dataclasses import dataclass, field, replace
from typing import Dict, List, Optional, Tuple

import numpy as np

from .bf16 import f32_to_bf16_bits

TARGETS = ("q", "k", "v", "o", "gate", "up", "down")


@dataclass(frozen=True)
class BackboneSpec:
    name: str
    n_layers: int
    d_model: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    d_ffn: int
    act: str            # 'gelu' (erf form) | 'relu' | 'swiglu'
    norm: str           # 'ln' | 'rms'
    norm_eps: float
    causal: bool
    rope_theta: float   # 0 = no RoPE
    input_kind: str     # 'embedded' | 'patch' | 'tokens'
    patch_dim: int = 0          # values per patch (patch kinds)
    tokens_per_request: int = 0  # 0 = variable length
    has_cls: bool = False
    vocab: int = 0
    max_seq: int = 0
    has_bias: bool = False
    # image geometry for patch kinds fed with raw images (0 = input is already [n_patch, patch_dim])
    img_c: int = 0
    img_hw: int = 0
    patch_hw: int = 0
    # generator-only knobs (distribution parameters)
    std: float = 0.02
    std_out: float = 0.02       # o and down projections
    std_embed: float = 0.02     # token table
    pos_kind: str = "none"      # 'none' | 'sinusoid' | 'normal'
    # NEXT-4 variant: T5-style relative-position bias, one table [rel_buckets, n_q_heads] shared by every layer (0 = none)
    rel_buckets: int = 0
    rel_max_distance: int = 0

    @property
    def d_q(self):
        return self.n_q_heads * self.head_dim

    @property
    def d_kv(self):
        return self.n_kv_heads * self.head_dim

    @property
    def n_patches(self):
        return self.tokens_per_request - (1 if self.has_cls else 0)


def target_dims(bb: BackboneSpec, target: str) -> Tuple[int, int]:
    """(d_in, d_out) of a LoRA target projection."""
    return {
        "q": (bb.d_model, bb.d_q), "k": (bb.d_model, bb.d_kv), "v": (bb.d_model, bb.d_kv),
        "o": (bb.d_q, bb.d_model), "gate": (bb.d_model, bb.d_ffn), "up": (bb.d_model, bb.d_ffn),
        "down": (bb.d_ffn, bb.d_model),
    }[target]


@dataclass(frozen=True)
class AdapterSpec:
    target: str
    rank: int
    alpha: float

    @property
    def scaling(self):
        return self.alpha / self.rank


@dataclass(frozen=True)
class TaskSpec:
    adapters: Tuple[AdapterSpec, ...]
    head_kind: str      # 'mean' | 'cls' | 'last' | 'flatten' | 'dense' (per token: output [n_i, head_out])
    head_out: int
    head_std: float = 0.02
    enc_channels: int = 0  # > 1: per-task input encoder, a linear channel combiner C -> 1 (Listing 2)
    head_hidden: int = 0   # > 0: MLP decoder head  W2 relu(W feat + b) + b2  (Listing 2, MLPDecoder hidden_dim)

    def d_feat(self, bb: BackboneSpec) -> int:
        return bb.d_model * bb.tokens_per_request if self.head_kind == "flatten" else bb.d_model


def _stream(seed: int, name: str) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[seed, zlib.crc32(name.encode())]))


def _zipf_ids(rng, n, T, s):
    """P(id = k-1) ∝ k^-s, inverse-CDF sampling (reading #17)."""
    w = np.arange(1, T + 1, dtype=np.float64) ** (-s)
    cdf = np.cumsum(w) / np.sum(w)
    u = rng.random(n)
    return np.minimum(np.searchsorted(cdf, u, side="right"), T - 1).astype(np.int32)


@dataclass
class Workload:
    cfg: str
    seed: int
    bb: BackboneSpec
    tasks: List[TaskSpec]
    task_ids: np.ndarray     # int32 [B], original request order
    lengths: np.ndarray      # int32 [B]
    notes: Dict[str, object] = field(default_factory=dict)
    lora_std: float = 0.02   # std of A and B draws (configs state 0.02; tests may stress it)

    # ---- tensors -------------------------------------------------------------------
    def shape_of(self, name: str) -> Tuple[int, ...]:
        return self._recipe(name)[0]

    def _recipe(self, name: str):
        """-> (shape, kind, std) ; kind in normal|gain|sinusoid."""
        bb = self.bb
        parts = name.split(".")
        if parts[0] == "embed":
            what = parts[1]
            if what == "W":
                return (bb.d_model, bb.patch_dim), "normal", bb.std
            if what == "b":
                return (bb.d_model,), "normal", bb.std
            if what == "cls":
                return (bb.d_model,), "normal", bb.std
            if what == "pos":
                return (bb.tokens_per_request, bb.d_model), bb.pos_kind, bb.std
            if what == "table":
                return (bb.vocab, bb.d_model), "normal", bb.std_embed
        if parts[0] == "rel_bias":         # NEXT-4 variant: T5 relative-position bias table [buckets, heads]; O(1) values so that it matters
            return (bb.rel_buckets, bb.n_q_heads), "normal", 1.0
        if parts[0] == "lm_head":          # NEXT-3: untied language-model head [vocab, d_model] (reading 34)
            return (bb.vocab, bb.d_model), "normal", 0.02
        if parts[0] == "final":
            return (bb.d_model,), ("gain" if parts[1] == "g" else "normal"), bb.std
        if parts[0].startswith("L") and len(parts[0]) == 3:
            what = parts[1]
            if what in ("norm1", "norm2"):
                return (bb.d_model,), ("gain" if parts[2] == "g" else "normal"), bb.std
            wshape = {"Wq": (bb.d_q, bb.d_model), "Wk": (bb.d_kv, bb.d_model),
                      "Wv": (bb.d_kv, bb.d_model), "Wo": (bb.d_model, bb.d_q),
                      "Wup": (bb.d_ffn, bb.d_model), "Wgate": (bb.d_ffn, bb.d_model),
                      "Wdown": (bb.d_model, bb.d_ffn)}
            if what in wshape:
                std = bb.std_out if what in ("Wo", "Wdown") else bb.std
                return wshape[what], "normal", std
            bshape = {"bq": bb.d_q, "bk": bb.d_kv, "bv": bb.d_kv, "bo": bb.d_model,
                      "bup": bb.d_ffn, "bgate": bb.d_ffn, "bdown": bb.d_model}
            if what in bshape:
                return (bshape[what],), "normal", bb.std
        if parts[0].startswith("task"):
            t = int(parts[0][4:])
            ts = self.tasks[t]
            if parts[1] == "enc":
                return ((ts.enc_channels,) if parts[2] == "W" else (1,)), "normal", (0.6 if parts[2] == "W" else 0.05)
            if parts[1] == "head":
                w1 = ts.head_hidden or ts.head_out                      # rows of the first (or only) layer
                if parts[2] == "W":
                    return (w1, ts.d_feat(bb)), "normal", ts.head_std
                if parts[2] == "W2":
                    return (ts.head_out, ts.head_hidden), "normal", 0.1
                if parts[2] == "b2":
                    return (ts.head_out,), "normal", 0.02
                return (w1,), "normal", 0.02
            tgt, ab = parts[2], parts[3]
            ad = next(a for a in ts.adapters if a.target == tgt)
            d_in, d_out = target_dims(bb, tgt)
            return ((ad.rank, d_in) if ab == "A" else (d_out, ad.rank)), "normal", self.lora_std
        raise KeyError(name)

    def tensor(self, name: str) -> np.ndarray:
        """bf16 bit patterns (uint16) of the named weight tensor; deterministic per (seed, name)."""
        shape, kind, std = self._recipe(name)
        if kind == "sinusoid":
            n, d = shape
            p = np.arange(n, dtype=np.float64)[:, None]
            div = np.exp(np.arange(0, d, 2, dtype=np.float64) * (-math.log(10000.0) / d))
            pe = np.zeros((n, d), dtype=np.float64)
            pe[:, 0::2] = np.sin(p * div)
            pe[:, 1::2] = np.cos(p * div)
            return f32_to_bf16_bits(pe.astype(np.float32))
        rng = _stream(self.seed, name)
        x = rng.standard_normal(shape, dtype=np.float32) * np.float32(std)
        if kind == "gain":
            x = np.float32(1.0) + x
        return f32_to_bf16_bits(x)

    # ---- per-request inputs --------------------------------------------------------
    def request_input(self, i: int) -> np.ndarray:
        """Input of request i in the form the C-ABI takes (uint16 bf16 bits, or int32 ids)."""
        bb = self.bb
        rng = _stream(self.seed, f"input.{i}")
        if bb.input_kind == "embedded":
            return f32_to_bf16_bits(rng.standard_normal((int(self.lengths[i]), bb.d_model),
                                                        dtype=np.float32))
        if bb.input_kind == "tokens":
            return rng.integers(0, bb.vocab, size=int(self.lengths[i]), dtype=np.int32)
        if bb.img_c:       # raw image, values U(0,1)
            return f32_to_bf16_bits(rng.random((bb.img_c, bb.img_hw, bb.img_hw), dtype=np.float32))
        # univariate random walk, z-normalised with the population std (reading #21); a task with an input encoder brings
        # C such channels, channel-major [C, n]
        n = bb.n_patches * bb.patch_dim
        C = max(self.tasks[int(self.task_ids[i])].enc_channels, 1)
        walk = np.cumsum(rng.standard_normal((C, n), dtype=np.float64), axis=1)
        z = (walk - walk.mean(axis=1, keepdims=True)) / walk.std(axis=1, keepdims=True)
        z = z[0] if C == 1 else z
        return f32_to_bf16_bits(z.astype(np.float32))

    def packed_inputs(self) -> np.ndarray:
        """All requests' inputs concatenated in ORIGINAL request order (flat array)."""
        return np.concatenate([self.request_input(i).reshape(-1) for i in range(len(self.task_ids))])

    # ---- names ---------------------------------------------------------------------
    def backbone_tensor_names(self) -> List[str]:
        bb = self.bb
        names = []
        if bb.input_kind == "patch":
            names += ["embed.W", "embed.b"]
            if bb.has_cls:
                names.append("embed.cls")
        if bb.input_kind == "tokens":
            names.append("embed.table")
        if bb.pos_kind != "none":
            names.append("embed.pos")
        if bb.rel_buckets:
            names.append("rel_bias.W")
        for l in range(bb.n_layers):
            names += self.layer_tensor_names(l)
        names.append("final.g")
        if bb.norm == "ln":
            names.append("final.b")
        return names

    def layer_tensor_names(self, l: int) -> List[str]:
        bb = self.bb
        p = f"L{l:02d}."
        ws = ["Wq", "Wk", "Wv", "Wo", "Wup", "Wdown"] + (["Wgate"] if bb.act == "swiglu" else [])
        names = [p + w for w in ws] + [p + "norm1.g", p + "norm2.g"]
        if bb.norm == "ln":
            names += [p + "norm1.b", p + "norm2.b"]
        if bb.has_bias:
            names += [p + "b" + w[1:] for w in ws]
        return names

    def task_tensor_names(self, t: int) -> List[str]:
        ts = self.tasks[t]
        names = [f"task{t:03d}.head.W", f"task{t:03d}.head.b"]
        if self.tasks[t].head_hidden:
            names += [f"task{t:03d}.head.W2", f"task{t:03d}.head.b2"]
        if self.tasks[t].enc_channels > 1:
            names += [f"task{t:03d}.enc.W", f"task{t:03d}.enc.b"]
        for l in range(self.bb.n_layers):
            for ad in ts.adapters:
                names += [f"task{t:03d}.L{l:02d}.{ad.target}.A", f"task{t:03d}.L{l:02d}.{ad.target}.B"]
        return names

    # ---- bookkeeping ---------------------------------------------------------------
    @property
    def n_req(self):
        return len(self.task_ids)

    @property
    def n_tokens(self):
        return int(np.sum(self.lengths))

    def out_offsets(self) -> np.ndarray:
        o = np.array([self.tasks[t].head_out * (int(n) if self.tasks[t].head_kind == "dense" else 1)
                      for t, n in zip(self.task_ids, self.lengths)], dtype=np.int64)
        return np.concatenate([[0], np.cumsum(o)])


# =====================================================================================
_BACKBONES = {
    "cfg1": BackboneSpec("tiny-encoder", 2, 128, 4, 4, 32, 512, "gelu", "ln", 1e-5, False, 0.0,
                         "embedded", tokens_per_request=64, max_seq=64, has_bias=True),
    "cfg2": BackboneSpec("t5-large-enc-shaped", 24, 1024, 16, 16, 64, 4096, "relu", "rms", 1e-6,
                         False, 0.0, "patch", patch_dim=8, tokens_per_request=64, max_seq=64,
                         has_bias=False, pos_kind="sinusoid"),
    "cfg3": BackboneSpec("vit-l14-shaped", 24, 1024, 16, 16, 64, 4096, "gelu", "ln", 1e-5, False,
                         0.0, "patch", patch_dim=588, tokens_per_request=257, has_cls=True,
                         max_seq=257, has_bias=True, img_c=3, img_hw=224, patch_hw=14,
                         pos_kind="normal"),
    "cfg4": BackboneSpec("decoder-lm-prefill", 28, 1536, 12, 2, 128, 8960, "swiglu", "rms", 1e-6,
                         True, 10000.0, "tokens", vocab=32000, max_seq=1024, has_bias=False,
                         std_out=0.02 / math.sqrt(56.0), std_embed=1.0),
}
_BACKBONES["cfg5"] = replace(_BACKBONES["cfg2"])
_RANKS5 = (4, 8, 16, 32, 64)
_DISTS = ("uniform", "zipf0.8", "zipf1.5")


def config_names():
    return ["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"]


def _tasks_for(cfg: str, seed: int, T: int) -> List[TaskSpec]:
    tasks = []
    for t in range(T):
        rng = _stream(seed, f"task{t:03d}.spec")
        if cfg == "cfg1":
            ads = tuple(AdapterSpec(x, 4, 8.0) for x in ("q", "v"))
            tasks.append(TaskSpec(ads, "mean", (5, 3, 10)[t % 3]))
        elif cfg == "cfg2":
            ads = tuple(AdapterSpec(x, 8, 16.0) for x in ("q", "k", "v", "o"))
            if t < 5:
                tasks.append(TaskSpec(ads, "flatten", 96, head_std=0.0025))
            else:
                tasks.append(TaskSpec(ads, "mean", int(rng.integers(2, 21))))
        elif cfg == "cfg3":
            r = (8, 16)[int(rng.integers(0, 2))]
            o = int(rng.integers(10, 1001))
            o = 1000 if t == 0 else (10 if t == 1 else o)     # reading #14: extremes forced
            ads = tuple(AdapterSpec(x, r, 16.0) for x in ("q", "k", "v", "o"))
            tasks.append(TaskSpec(ads, "cls", o))
        elif cfg == "cfg4":
            r = _RANKS5[int(rng.integers(0, 5))]
            o = 1 if t % 5 == 4 else int(rng.integers(2, 51))
            ads = tuple(AdapterSpec(x, r, 16.0) for x in TARGETS)
            tasks.append(TaskSpec(ads, "last", o))
        elif cfg == "cfg5":
            r = 16 if T == 1 else _RANKS5[int(rng.integers(0, 5))]
            ads = tuple(AdapterSpec(x, r, 16.0) for x in ("q", "k", "v", "o"))
            if T == 1 or t % 2 == 0:
                tasks.append(TaskSpec(ads, "flatten", 96, head_std=0.0025))
            else:
                tasks.append(TaskSpec(ads, "mean", int(rng.integers(2, 21))))
        else:
            raise KeyError(cfg)
    return tasks


def make_workload(cfg: str, *, n_layers: Optional[int] = None, batch: Optional[int] = None,
                  n_tasks: Optional[int] = None, dist: Optional[str] = None,
                  max_len: Optional[int] = None, adapters: bool = True,
                  seed_offset: int = 0, lora_std: float = 0.02, mlp_hidden: int = 0,
                  enc_channels: int = 0, dense_heads: bool = False, rel_bias: bool = False) -> Workload:
    """Build the workload of a BASELINE.json config (cfg1..cfg5).

    Overrides give the reduced variants the parity tests use (fewer layers, smaller batch);
    with no overrides the result is the full config.  cfg5 takes n_tasks in {1,4,16,48,92}
    and dist in {'uniform','zipf0.8','zipf1.5'}; adapters=False registers head-only tasks
    (the adapter-free reference of reading #19).  lora_std != 0.02 is a STRESS variant for
    tests that need the adapter delta to dominate the tolerance; it is not a config.  mlp_hidden > 0 turns
    every pooled (non-flatten) head into an MLP decoder head of that hidden width (the
    paper's Listing 2 uses hidden_dim 128) - a test variant, not a BASELINE.json config.
    """
    bb = _BACKBONES[cfg]
    if n_layers is not None:
        bb = replace(bb, n_layers=n_layers)
    if rel_bias:            # the T5 relative-position bias (32 buckets, max distance 128: T5's defaults); a variant
        bb = replace(bb, rel_buckets=32, rel_max_distance=128)
    idx = int(cfg[3])
    seed = 9643000 + idx + seed_offset
    defaults = {"cfg1": (12, 3), "cfg2": (256, 10), "cfg3": (128, 32), "cfg4": (64, 92),
                "cfg5": (512, 92)}
    B = batch if batch is not None else defaults[cfg][0]
    T = n_tasks if n_tasks is not None else defaults[cfg][1]
    if cfg == "cfg5":
        dist = dist or "zipf0.8"
        seed += 100 * T + 10 * _DISTS.index(dist)
    tasks = _tasks_for(cfg, seed, T)
    if not adapters:
        tasks = [replace(t, adapters=()) for t in tasks]
    if mlp_hidden:
        tasks = [t if t.head_kind == "flatten" else replace(t, head_hidden=mlp_hidden) for t in tasks]
    if dense_heads:               # test variant (NEXT-1): every third task decodes EVERY token (dense / segmentation-style head)
        tasks = [replace(t, head_kind="dense", head_hidden=0, head_std=0.02, head_out=min(t.head_out, 21)) if i % 3 == 1 else t
                 for i, t in enumerate(tasks)]
    if enc_channels > 1:          # test variant (NEXT-1): every other task brings enc_channels input channels and a combiner
        tasks = [replace(t, enc_channels=enc_channels) if i % 2 == 0 else t for i, t in enumerate(tasks)]
    rng = _stream(seed, "task_ids")
    if cfg == "cfg1":
        while True:                                   # reading #20: every task present
            ids = rng.integers(0, T, size=B).astype(np.int32)
            if B < T or len(np.unique(ids)) == T:
                break
    elif cfg == "cfg2":
        ids = _zipf_ids(rng, B, T, 1.1)
    elif cfg == "cfg3":
        ids = rng.integers(0, T, size=B).astype(np.int32)
    elif cfg == "cfg4":
        ids = _zipf_ids(rng, B, T, 1.0)
    else:                                             # cfg5, reading #18: every task present
        n_free = max(B - T, 0)
        if dist == "uniform":
            rest = rng.integers(0, T, size=n_free).astype(np.int32)
        else:
            rest = _zipf_ids(rng, n_free, T, float(dist[4:]))
        ids = np.concatenate([np.arange(min(T, B), dtype=np.int32), rest])
        ids = ids[rng.permutation(len(ids))].astype(np.int32)
    if bb.tokens_per_request:
        lengths = np.full(B, bb.tokens_per_request, dtype=np.int32)
    else:
        hi = min(max_len or bb.max_seq, bb.max_seq)
        lo = min(64, hi)
        lengths = _stream(seed, "lengths").integers(lo, hi + 1, size=B).astype(np.int32)
    return Workload(cfg, seed, bb, tasks, ids, lengths, notes={"dist": dist}, lora_std=lora_std)
