"""ORACLE (test infrastructure, not product code) — the vFM forward, by definition, in fp64.

What it is.  FMplex gives every task a *virtual foundation model*: "the illusion that it is
running exclusively on its own foundation model" (§4.1), i.e. the shared
backbone plus that task's PEFT adapter plus that task's decoder head (PAPER.md L119-L120
"Task Extensions"; L76 "executes each task's requests ... against the shared backbone and
then applies the task-specific decoder head"; L174 adapters are "applied internally during
the forward pass").  A mixed batch is therefore *defined* as: every request alone through
its own model.  This file evaluates exactly that, one request at a time, in numpy float64,
with no batching across requests, no sorting, no segment tables and no tiling.  The CUDA
path shares no code with it, and nothing under the product package imports it.

LoRA form (PEFT `LoraConfig(r, lora_alpha, target_modules)`, Listing 2):
    Lin_P(x) = x W_P^T + b_P + (alpha/r) (x A^T) B^T.
Architectural details (norm kinds, activations, RoPE, GQA, pooling) are those BASELINE.json
`configs` names; the readings of everything the paper leaves open are DESIGN.md §3.

Inputs are plain numpy arrays fetched through a caller-supplied `get(name)` that returns
float64 arrays (the bf16-rounded values the GPU receives, widened).  Tensor names:
    embed.W [d,patch_dim]  embed.b [d]  embed.cls [d]  embed.pos [n_pos,d]  embed.table [vocab,d]
    L{ll}.norm1.g/.b  L{ll}.Wq/.Wk/.Wv/.Wo/.Wup/.Wgate/.Wdown  L{ll}.bq/... (if bias)
    L{ll}.norm2.g/.b  final.g/.b
    task{ttt}.L{ll}.{target}.A [r,d_in]  .B [d_out,r]   task{ttt}.head.W [o,d_feat]  .head.b [o]
`bb` is a dict of hyper-parameters (see `REQUIRED_BB_KEYS`); `task` is a dict
{id, adapters: {target: (rank, scaling)}, head_kind, head_out[, head_hidden]}.

Pins (tests/test_oracle_pins.py): brute-force matmul on tiny shapes; closed forms for the
norms, softmax, GeLU/SiLU, RoPE; the LoRA merge identity W' = W + s·B·A; zero adapter ==
backbone-only; pooling/flatten special cases; a hand-expanded 1-layer, 2-token, d=2 example.
Library pins (tests/test_oracle_library_pins.py, independent PyTorch / Hugging Face code in fp64):
`attention` vs torch SDPA (causal / full, GQA); the norms and activations vs torch.nn.functional;
`layer_forward` of both encoder families vs torch.nn.TransformerEncoderLayer(norm_first=True);
the decoder backbone (RMSNorm, rotate-half RoPE, GQA, causal, SwiGLU) with LoRA on all seven
targets vs transformers' LlamaModel carrying the merged weights W + (alpha/r) B A; the relative-position bias variant
(`rel_bucket`, NEXT-4) vs transformers' T5Attention bucket function and a whole T5Block, plus hand-derived bucket values.
The paper prints no value of any forward output, so no pin comes from the paper itself; what
stays without a library counterpart is only the pooled / flattened head (a mean, a row pick or
a reshape, then one matrix-vector product), pinned by its special cases; the
image patch embedding is pinned against torch.nn.Conv2d.
"""
import math

import numpy as np
from scipy.special import erf as _erf   # library primitive; pinned against math.erf in tests

REQUIRED_BB_KEYS = ("n_layers", "d_model", "n_q_heads", "n_kv_heads", "head_dim", "d_ffn", "act",
                    "norm", "norm_eps", "causal", "rope_theta", "input_kind", "patch_dim",
                    "has_cls", "has_bias", "has_pos", "img_c", "img_hw", "patch_hw")


# ---------------------------------------------------------------- elementary pieces
def brute_matmul(a, b):
    """Triple-loop matrix product in Python floats (pin for `@` on tiny shapes)."""
    n, k = len(a), len(a[0])
    m = len(b[0])
    out = [[0.0] * m for _ in range(n)]
    for i in range(n):
        for j in range(m):
            s = 0.0
            for p in range(k):
                s += float(a[i][p]) * float(b[p][j])
            out[i][j] = s
    return np.array(out, dtype=np.float64)


def layer_norm(x, g, b, eps):
    """(x-mu)/sqrt(var+eps)*g + b, biased variance over the last axis."""
    mu = x.mean(axis=-1, keepdims=True)
    var = ((x - mu) ** 2).mean(axis=-1, keepdims=True)
    return (x - mu) / np.sqrt(var + eps) * g + b


def rms_norm(x, g, eps):
    """x/sqrt(mean(x^2)+eps)*g over the last axis."""
    return x / np.sqrt((x * x).mean(axis=-1, keepdims=True) + eps) * g


def gelu_erf(x):
    return 0.5 * x * (1.0 + _erf(x / math.sqrt(2.0)))


def silu(x):
    return x / (1.0 + np.exp(-x))


def relu(x):
    return np.maximum(x, 0.0)


def softmax_rows(s):
    m = s.max(axis=-1, keepdims=True)
    e = np.exp(s - m)
    return e / e.sum(axis=-1, keepdims=True)


def rope_rotate_half(x, theta):
    """x [n, d_h]; position p = row index within the request (0-based); rotate-half pairing
    (j, j+d_h/2), angle p * theta^(-2j/d_h)  (DESIGN.md §3 reading 7)."""
    n, dh = x.shape
    half = dh // 2
    inv = theta ** (-2.0 * np.arange(half, dtype=np.float64) / dh)
    ang = np.arange(n, dtype=np.float64)[:, None] * inv[None, :]
    c, s = np.cos(ang), np.sin(ang)
    x1, x2 = x[:, :half], x[:, half:]
    return np.concatenate([x1 * c - x2 * s, x2 * c + x1 * s], axis=1)


def attention(q, k, v, n_q_heads, n_kv_heads, head_dim, causal, bias=None):
    """softmax(q k^T / sqrt(d_h) + M + bias_g) v per query head; query head g reads KV head
    floor(g / (H_q/H_kv)); M_ab = -inf for b > a when causal; bias: None or [H_q, n, n] added to the scores."""
    n = q.shape[0]
    group = n_q_heads // n_kv_heads
    out = np.empty((n, n_q_heads * head_dim), dtype=np.float64)
    for g in range(n_q_heads):
        kv = g // group
        qg = q[:, g * head_dim:(g + 1) * head_dim]
        kg = k[:, kv * head_dim:(kv + 1) * head_dim]
        vg = v[:, kv * head_dim:(kv + 1) * head_dim]
        s = (qg @ kg.T) / math.sqrt(head_dim)
        if bias is not None:
            s = s + bias[g]
        if causal:
            s = np.where(np.arange(n)[None, :] > np.arange(n)[:, None], -np.inf, s)
        out[:, g * head_dim:(g + 1) * head_dim] = softmax_rows(s) @ vg
    return out


def rel_bucket(rel, bidirectional, n_buckets, max_distance):
    """Bucket of the relative position rel = key position - query position (T5: Raffel et al. 2020, section 2.1 "we use 32
    embeddings ... with ranges that increase in size logarithmically up to an offset of 128 beyond which we assign all relative
    positions to the same embedding").  Step by step:
      bidirectional (encoder): half of the buckets for keys after the query (rel > 0), half for keys at or before it; the
        distance is |rel|.  Unidirectional (causal): keys after the query all map to distance 0; the distance is max(-rel, 0).
      Of the n buckets on a side the first n / 2 hold the distances 0 .. n/2 - 1 exactly; the other n / 2 hold logarithmically
        growing ranges up to max_distance, everything beyond falls in the last bucket:
        n/2 + floor( log(dist / (n/2)) / log(max_distance / (n/2)) * (n - n/2) ), capped at n - 1."""
    rel = int(rel)
    n = n_buckets
    b = 0
    if bidirectional:
        n //= 2
        if rel > 0:
            b += n
        dist = abs(rel)
    else:
        dist = max(-rel, 0)
    max_exact = n // 2
    if dist < max_exact:
        return b + dist
    large = max_exact + int(math.log(dist / max_exact) / math.log(max_distance / max_exact) * (n - max_exact))
    return b + min(large, n - 1)


def rel_bias_matrix(table, n, bidirectional, n_buckets, max_distance):
    """bias[g, a, b] = table[rel_bucket(b - a), g] for query position a, key position b; table [n_buckets, H_q]."""
    H = table.shape[1]
    out = np.empty((H, n, n), dtype=np.float64)
    for a in range(n):
        for b in range(n):
            out[:, a, b] = table[rel_bucket(b - a, bidirectional, n_buckets, max_distance)]
    return out


def lora_linear(x, W, b, adapter):
    """x W^T + b + s (x A^T) B^T ; adapter = None or (A [r,d_in], B [d_out,r], s)."""
    y = x @ W.T
    if b is not None:
        y = y + b
    if adapter is not None:
        A, B, s = adapter
        y = y + s * ((x @ A.T) @ B.T)
    return y


# ---------------------------------------------------------------- the definition
def tokens_from_input(bb, get, x, task=None):
    """Step 1: request input -> h0 [n, d].  A task with an input encoder (Listing 2,
    LinearChannelCombiner(num_channels = C, new_num_channels = 1)) first maps its C channels to the one series the backbone
    takes: sum_c w[c] x[c, :] + b."""
    kind = bb["input_kind"]
    if task is not None and task.get("enc_channels", 0) > 1:
        C = task["enc_channels"]
        p = f"task{task['id']:03d}.enc."
        x = get(p + "W") @ np.asarray(x, dtype=np.float64).reshape(C, -1) + get(p + "b")[0]
    if kind == "embedded":
        return np.array(x, dtype=np.float64)
    if kind == "tokens":
        return get("embed.table")[np.asarray(x, dtype=np.int64)]
    # patch-linear
    if bb["img_c"]:
        C, HW, P = bb["img_c"], bb["img_hw"], bb["patch_hw"]
        g = HW // P
        img = np.asarray(x, dtype=np.float64).reshape(C, HW, HW)
        rows = []
        for gy in range(g):              # patches row-major over the grid,
            for gx in range(g):          # each flattened in (channel, row, col) order
                rows.append(img[:, gy * P:(gy + 1) * P, gx * P:(gx + 1) * P].reshape(-1))
        patches = np.stack(rows)
    else:
        patches = np.asarray(x, dtype=np.float64).reshape(-1, bb["patch_dim"])
    h = patches @ get("embed.W").T + get("embed.b")
    if bb["has_cls"]:
        h = np.concatenate([get("embed.cls")[None, :], h], axis=0)
    if bb["has_pos"]:
        h = h + get("embed.pos")[:h.shape[0]]
    return h


def _norm(bb, get, prefix, x):
    if bb["norm"] == "ln":
        return layer_norm(x, get(prefix + ".g"), get(prefix + ".b"), bb["norm_eps"])
    return rms_norm(x, get(prefix + ".g"), bb["norm_eps"])


def _adapter(get, task, l, target):
    if task is None or target not in task["adapters"]:
        return None
    _rank, s = task["adapters"][target]
    p = f"task{task['id']:03d}.L{l:02d}.{target}."
    return get(p + "A"), get(p + "B"), s


def layer_forward(bb, get, task, l, h, capture=None):
    """Step 2 for one layer (pre-norm), one request."""
    p = f"L{l:02d}."
    bias = (lambda n: get(p + n)) if bb["has_bias"] else (lambda n: None)
    a = _norm(bb, get, p + "norm1", h)
    q = lora_linear(a, get(p + "Wq"), bias("bq"), _adapter(get, task, l, "q"))
    k = lora_linear(a, get(p + "Wk"), bias("bk"), _adapter(get, task, l, "k"))
    v = lora_linear(a, get(p + "Wv"), bias("bv"), _adapter(get, task, l, "v"))
    Hq, Hkv, dh = bb["n_q_heads"], bb["n_kv_heads"], bb["head_dim"]
    if bb["rope_theta"] > 0:
        q = np.concatenate([rope_rotate_half(q[:, g * dh:(g + 1) * dh], bb["rope_theta"])
                            for g in range(Hq)], axis=1)
        k = np.concatenate([rope_rotate_half(k[:, g * dh:(g + 1) * dh], bb["rope_theta"])
                            for g in range(Hkv)], axis=1)
    rel = None
    if bb.get("rel_buckets", 0) > 0:        # one table for every layer, as in T5 (the first block owns it, the others reuse it)
        rel = rel_bias_matrix(get("rel_bias.W"), h.shape[0], not bb["causal"], bb["rel_buckets"], bb["rel_max_distance"])
    o = attention(q, k, v, Hq, Hkv, dh, bb["causal"], rel)
    h = h + lora_linear(o, get(p + "Wo"), bias("bo"), _adapter(get, task, l, "o"))
    m = _norm(bb, get, p + "norm2", h)
    if bb["act"] == "swiglu":
        gate = lora_linear(m, get(p + "Wgate"), bias("bgate"), _adapter(get, task, l, "gate"))
        up = lora_linear(m, get(p + "Wup"), bias("bup"), _adapter(get, task, l, "up"))
        hid = silu(gate) * up
    else:
        up = lora_linear(m, get(p + "Wup"), bias("bup"), _adapter(get, task, l, "up"))
        hid = gelu_erf(up) if bb["act"] == "gelu" else relu(up)
    if capture is not None:
        capture.update(norm1=a, q=q, k=k, v=v, attn=o, norm2=m, hid=hid)
    return h + lora_linear(hid, get(p + "Wdown"), bias("bdown"), _adapter(get, task, l, "down"))


def pooled_feature(f, head_kind):
    """Step 4."""
    if head_kind == "mean":
        return f.mean(axis=0)
    if head_kind == "cls":
        return f[0]
    if head_kind == "last":
        return f[-1]
    if head_kind == "flatten":
        return f.reshape(-1)          # token-major, then channel
    raise ValueError(head_kind)


def head_forward(bb, get, task, h):
    """Steps 3-5: final norm, pool, linear head."""
    f = _norm(bb, get, "final", h)
    p = f"task{task['id']:03d}.head."
    if task["head_kind"] == "dense":
        # dense (per-token) decoder, "dense decoders for ... detection, and segmentation" (
        # DESIGN.md reading 35): the head is applied to EVERY token row; the output is [n, o_t] row-major (token, then class)
        return (f @ get(p + "W").T + get(p + "b")).reshape(-1)
    feat = pooled_feature(f, task["head_kind"])
    y = get(p + "W") @ feat + get(p + "b")
    if task.get("head_hidden", 0):
        # MLP decoder head (Listing 2: MLPDecoder(input_dim, hidden_dim, output_dim)); the paper names the three
        # widths only - ReLU between the two linear layers is DESIGN.md reading 32
        y = get(p + "W2") @ relu(y) + get(p + "b2")
    return y


def forward_request(bb, get, task, x):
    """The vFM forward of ONE request: backbone + its task's adapter + its task's head."""
    h = tokens_from_input(bb, get, x, task)
    for l in range(bb["n_layers"]):
        h = layer_forward(bb, get, task, l, h)
    return head_forward(bb, get, task, h)


def forward_requests(bb, get, tasks, task_ids, inputs):
    """Every request separately; the layer loop is outermost only so that a caller's `get`
    may widen one layer's weights at a time (each request's arithmetic is untouched)."""
    hs = [tokens_from_input(bb, get, x, tasks[t]) for x, t in zip(inputs, task_ids)]
    for l in range(bb["n_layers"]):
        hs = [layer_forward(bb, get, tasks[t], l, h) for h, t in zip(hs, task_ids)]
    return [head_forward(bb, get, tasks[t], h) for h, t in zip(hs, task_ids)]
