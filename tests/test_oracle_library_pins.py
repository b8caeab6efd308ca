"""Pins of the oracle against INDEPENDENT library implementations of the same textbook models (fp64, CPU):

* `attention`              vs torch.nn.functional.scaled_dot_product_attention (causal / full, GQA by repeating KV heads)
* `layer_norm`, `rms_norm`,
  `gelu_erf`, `silu`        vs torch.nn.functional
* `layer_forward` of both encoder families (pre-LN + GeLU + biases: cfg1 / cfg3; RMSNorm + ReLU, no biases: cfg2 / cfg5)
                            vs torch.nn.TransformerEncoderLayer(norm_first=True) carrying the same weights
* the whole backbone of the decoder family (RMSNorm, rotate-half RoPE, GQA, causal, SwiGLU: cfg4) WITH per-task LoRA
                            vs transformers' LlamaModel carrying the merged weights W + (alpha/r) B A

The oracle is numpy, these are PyTorch / Hugging Face code written by other people: a wrong sign in RoPE, a transposed
operand, a head-grouping mistake, a mis-placed adapter or norm fails here.  None of this touches the CUDA path.
"""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
F = torch.nn.functional

from oracle import vfm_forward as O  # noqa: E402

T64 = dict(dtype=torch.float64)


def _rng(seed):
    return np.random.default_rng(seed)


def _t(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(torch.float64)


# ---------------------------------------------------------------- elementary pieces
@pytest.mark.parametrize("causal", [0, 1])
@pytest.mark.parametrize("hq,hkv,dh,n", [(4, 4, 8, 13), (6, 2, 16, 37), (8, 1, 4, 5), (3, 3, 32, 1)])
def test_attention_matches_torch_sdpa(hq, hkv, dh, n, causal):
    r = _rng(hq * 100 + n)
    q, k, v = r.standard_normal((n, hq * dh)), r.standard_normal((n, hkv * dh)), r.standard_normal((n, hkv * dh))
    got = O.attention(q, k, v, hq, hkv, dh, bool(causal))
    tq = _t(q).view(n, hq, dh).transpose(0, 1)                                   # [H, n, dh]
    tk = _t(k).view(n, hkv, dh).transpose(0, 1).repeat_interleave(hq // hkv, dim=0)
    tv = _t(v).view(n, hkv, dh).transpose(0, 1).repeat_interleave(hq // hkv, dim=0)
    ref = F.scaled_dot_product_attention(tq[None], tk[None], tv[None], is_causal=bool(causal))[0]
    ref = ref.transpose(0, 1).reshape(n, hq * dh).numpy()
    assert np.allclose(got, ref, rtol=1e-11, atol=1e-12)


def test_norms_and_activations_match_torch():
    r = _rng(7)
    x, g, b = r.standard_normal((9, 24)) * 3, r.standard_normal(24), r.standard_normal(24)
    assert np.allclose(O.layer_norm(x, g, b, 1e-5), F.layer_norm(_t(x), (24,), _t(g), _t(b), 1e-5).numpy(), rtol=1e-12, atol=1e-13)
    if hasattr(F, "rms_norm"):
        assert np.allclose(O.rms_norm(x, g, 1e-6), F.rms_norm(_t(x), (24,), _t(g), 1e-6).numpy(), rtol=1e-12, atol=1e-13)
    y = np.linspace(-9, 9, 1001)
    assert np.allclose(O.gelu_erf(y), F.gelu(_t(y), approximate="none").numpy(), rtol=1e-12, atol=1e-14)
    assert np.allclose(O.silu(y), F.silu(_t(y)).numpy(), rtol=1e-12, atol=1e-14)
    assert np.allclose(O.relu(y), F.relu(_t(y)).numpy())


# ---------------------------------------------------------------- encoder families vs nn.TransformerEncoderLayer
@pytest.mark.parametrize("norm,act,has_bias", [("ln", "gelu", True),      # cfg1 / cfg3: pre-LayerNorm, exact GeLU, biases
                                               ("rms", "relu", False)])   # cfg2 / cfg5: RMSNorm, ReLU, no biases
def test_pre_norm_layers_match_torch_transformer_encoder_layer(norm, act, has_bias):
    if norm == "rms" and not hasattr(torch.nn, "RMSNorm"):
        pytest.skip("torch.nn.RMSNorm not available")
    d, H, Fd, n, L = 32, 4, 80, 19, 2
    eps = 1e-5 if norm == "ln" else 1e-6
    r = _rng(2026)
    W = {}
    for l in range(L):
        p = f"L{l:02d}."
        for nm, shape in (("Wq", (d, d)), ("Wk", (d, d)), ("Wv", (d, d)), ("Wo", (d, d)), ("Wup", (Fd, d)), ("Wdown", (d, Fd))):
            W[p + nm] = r.standard_normal(shape) * 0.2
        for nm, m in (("bq", d), ("bk", d), ("bv", d), ("bo", d), ("bup", Fd), ("bdown", d)):
            W[p + nm] = r.standard_normal(m) * 0.1
        for nm in ("norm1", "norm2"):
            W[p + nm + ".g"] = 1 + 0.1 * r.standard_normal(d)
            W[p + nm + ".b"] = 0.1 * r.standard_normal(d)
    bb = dict(n_layers=L, d_model=d, n_q_heads=H, n_kv_heads=H, head_dim=d // H, d_ffn=Fd, act=act, norm=norm, norm_eps=eps,
              causal=False, rope_theta=0.0, input_kind="embedded", patch_dim=0, has_cls=False, has_bias=has_bias, has_pos=False,
              img_c=0, img_hw=0, patch_hw=0)
    x = r.standard_normal((n, d))
    h = x
    for l in range(L):
        h = O.layer_forward(bb, W.__getitem__, None, l, h)

    act_fn = (lambda z: F.gelu(z, approximate="none")) if act == "gelu" else F.relu
    ht = _t(x)[None]
    for l in range(L):
        p = f"L{l:02d}."
        layer = torch.nn.TransformerEncoderLayer(d, H, Fd, dropout=0.0, activation=act_fn, layer_norm_eps=eps, batch_first=True,
                                                 norm_first=True, bias=has_bias, **T64)
        if norm == "rms":
            layer.norm1 = torch.nn.RMSNorm(d, eps=eps, **T64)
            layer.norm2 = torch.nn.RMSNorm(d, eps=eps, **T64)
        with torch.no_grad():
            layer.self_attn.in_proj_weight.copy_(_t(np.concatenate([W[p + "Wq"], W[p + "Wk"], W[p + "Wv"]])))
            layer.self_attn.out_proj.weight.copy_(_t(W[p + "Wo"]))
            layer.linear1.weight.copy_(_t(W[p + "Wup"]))
            layer.linear2.weight.copy_(_t(W[p + "Wdown"]))
            layer.norm1.weight.copy_(_t(W[p + "norm1.g"]))
            layer.norm2.weight.copy_(_t(W[p + "norm2.g"]))
            if has_bias:
                layer.self_attn.in_proj_bias.copy_(_t(np.concatenate([W[p + "bq"], W[p + "bk"], W[p + "bv"]])))
                layer.self_attn.out_proj.bias.copy_(_t(W[p + "bo"]))
                layer.linear1.bias.copy_(_t(W[p + "bup"]))
                layer.linear2.bias.copy_(_t(W[p + "bdown"]))
            if norm == "ln":
                layer.norm1.bias.copy_(_t(W[p + "norm1.b"]))
                layer.norm2.bias.copy_(_t(W[p + "norm2.b"]))
        layer.train()                                        # dropout is 0; train mode keeps PyTorch off its fused fast path
        with torch.no_grad():
            ht = layer(ht)
    assert np.allclose(h, ht[0].numpy(), rtol=1e-10, atol=1e-11)


# ---------------------------------------------------------------- decoder family (+ LoRA) vs transformers' LlamaModel
def _llama_fixture(tr):
    """A 2-layer Llama-shaped decoder (RMSNorm, rotate-half RoPE, GQA 3:1, causal, SwiGLU) with one task's LoRA on all 7
    targets: the oracle's weight dict / task, and transformers' LlamaForCausalLM carrying the MERGED weights
    W + (alpha / r) B A and an untied LM head."""
    d, Hq, Hkv, dh, Fd, L, vocab = 48, 6, 2, 8, 80, 2, 61
    theta, eps = 10000.0, 1e-6
    r = _rng(9643)
    W = {"embed.table": r.standard_normal((vocab, d)), "final.g": 1 + 0.1 * r.standard_normal(d),
         "lm_head.W": r.standard_normal((vocab, d)) * 0.3}
    dims = dict(q=(d, Hq * dh), k=(d, Hkv * dh), v=(d, Hkv * dh), o=(Hq * dh, d), gate=(d, Fd), up=(d, Fd), down=(Fd, d))
    ranks = dict(q=4, k=2, v=8, o=3, gate=5, up=1, down=6)
    task = dict(id=7, adapters={tg: (ranks[tg], 16.0 / ranks[tg]) for tg in dims}, head_kind="last", head_out=3)
    for l in range(L):
        p = f"L{l:02d}."
        for tg, (din, dout) in dims.items():
            W[p + "W" + tg] = r.standard_normal((dout, din)) * 0.15
            W[f"task007.{p}{tg}.A"] = r.standard_normal((ranks[tg], din)) * 0.2
            W[f"task007.{p}{tg}.B"] = r.standard_normal((dout, ranks[tg])) * 0.2
        W[p + "norm1.g"] = 1 + 0.1 * r.standard_normal(d)
        W[p + "norm2.g"] = 1 + 0.1 * r.standard_normal(d)
    bb = dict(n_layers=L, d_model=d, n_q_heads=Hq, n_kv_heads=Hkv, head_dim=dh, d_ffn=Fd, act="swiglu", norm="rms", norm_eps=eps,
              causal=True, rope_theta=theta, input_kind="tokens", patch_dim=0, has_cls=False, has_bias=False, has_pos=False,
              img_c=0, img_hw=0, patch_hw=0)
    cfg = tr.LlamaConfig(vocab_size=vocab, hidden_size=d, intermediate_size=Fd, num_hidden_layers=L, num_attention_heads=Hq,
                         num_key_value_heads=Hkv, head_dim=dh, hidden_act="silu", max_position_embeddings=64, rms_norm_eps=eps,
                         rope_theta=theta, attention_bias=False, mlp_bias=False, attention_dropout=0.0, tie_word_embeddings=False)
    cfg._attn_implementation = "eager"
    lm = tr.LlamaForCausalLM(cfg).to(torch.float64).eval()
    model = lm.model
    # rotary tables are buffers built in fp32: rebuild them in fp64 so the comparison is not limited by them
    inv = 1.0 / (theta ** (torch.arange(0, dh, 2, dtype=torch.float64) / dh))
    model.rotary_emb.inv_freq = inv
    if hasattr(model.rotary_emb, "original_inv_freq"):
        model.rotary_emb.original_inv_freq = inv

    def merged(l, tg):
        p = f"L{l:02d}."
        s = task["adapters"][tg][1]
        return _t(W[p + "W" + tg] + s * W[f"task007.{p}{tg}.B"] @ W[f"task007.{p}{tg}.A"])

    with torch.no_grad():
        model.embed_tokens.weight.copy_(_t(W["embed.table"]))
        model.norm.weight.copy_(_t(W["final.g"]))
        lm.lm_head.weight.copy_(_t(W["lm_head.W"]))
        for l, layer in enumerate(model.layers):
            layer.self_attn.q_proj.weight.copy_(merged(l, "q")); layer.self_attn.k_proj.weight.copy_(merged(l, "k"))
            layer.self_attn.v_proj.weight.copy_(merged(l, "v")); layer.self_attn.o_proj.weight.copy_(merged(l, "o"))
            layer.mlp.gate_proj.weight.copy_(merged(l, "gate")); layer.mlp.up_proj.weight.copy_(merged(l, "up"))
            layer.mlp.down_proj.weight.copy_(merged(l, "down"))
            layer.input_layernorm.weight.copy_(_t(W[f"L{l:02d}.norm1.g"]))
            layer.post_attention_layernorm.weight.copy_(_t(W[f"L{l:02d}.norm2.g"]))
    return bb, W, task, lm, r


def test_decoder_backbone_with_lora_matches_hf_llama_with_merged_weights():
    tr = pytest.importorskip("transformers")
    bb, W, task, lm, r = _llama_fixture(tr)
    model, eps, n = lm.model, bb["norm_eps"], 23
    toks = r.integers(0, W["embed.table"].shape[0], size=n)
    h = O.tokens_from_input(bb, W.__getitem__, toks)
    for l in range(bb["n_layers"]):
        h = O.layer_forward(bb, W.__getitem__, task, l, h)
    got = O.rms_norm(h, W["final.g"], eps)                      # what head_forward pools from
    with torch.no_grad():
        out = model(input_ids=torch.from_numpy(np.asarray(toks, dtype=np.int64))[None]).last_hidden_state[0].numpy()
    # LlamaRotaryEmbedding evaluates cos / sin in fp32 whatever the model dtype, which bounds the agreement at ~1e-6 relative
    # per rotation (measured here: 5e-6 absolute on outputs of magnitude 3); any structural mistake is O(0.1 .. 1).
    err = np.abs(got - out).max()
    assert err < 5e-5 * max(1.0, np.abs(out).max()), f"oracle vs LlamaModel: max abs {err:.3e}"
    # sensitivity: the comparison really sees the adapters (an un-merged model differs by far more than the bar)
    with torch.no_grad():
        model.layers[0].self_attn.q_proj.weight.copy_(_t(W["L00.Wq"]))
        out2 = model(input_ids=torch.from_numpy(np.asarray(toks, dtype=np.int64))[None]).last_hidden_state[0].numpy()
    assert np.abs(got - out2).max() > 1e-3


def test_token_decode_matches_hf_llama_incremental_decoding_with_a_kv_cache():
    """oracle.decode recomputes the whole prefix for every new token - the definition.  transformers'
    LlamaForCausalLM decodes INCREMENTALLY: the prompt once, then one token per call against its key / value cache
    (`past_key_values`).  Both must give the same next-token scores at every step and the same greedy continuation: this
    pins the definition and, independently, the claim that a KV cache does not change it."""
    tr = pytest.importorskip("transformers")
    from oracle import decode as D
    bb, W, task, lm, r = _llama_fixture(tr)
    vocab = W["embed.table"].shape[0]
    prompt = r.integers(0, vocab, size=9)
    n_new = 7
    toks, scores = D.greedy_decode(bb, W.__getitem__, task, prompt, n_new)
    with torch.no_grad():
        out = lm(input_ids=torch.from_numpy(np.asarray(prompt, dtype=np.int64))[None], use_cache=True)
        past, hf_scores, hf_toks = out.past_key_values, [out.logits[0, -1].numpy()], []
        for s in range(n_new):
            nxt = int(np.argmax(hf_scores[-1]))
            hf_toks.append(nxt)
            if s + 1 < n_new:
                out = lm(input_ids=torch.tensor([[nxt]]), past_key_values=past, use_cache=True)
                past = out.past_key_values
                hf_scores.append(out.logits[0, -1].numpy())
    assert toks == hf_toks, f"greedy continuation differs: {toks} vs {hf_toks}"
    for s, (a, b) in enumerate(zip(scores, hf_scores)):
        err = np.abs(a - b).max()
        assert err < 5e-5 * max(1.0, np.abs(b).max()), f"step {s}: oracle vs incremental HF decode: max abs {err:.3e}"
    # the scores of a step are the LM head on the last row of the plain forward over the prefix (the definition, re-stated
    # with the forward's own pieces) and they DO depend on the adapters
    seq = list(prompt) + toks[:3]
    h = O.tokens_from_input(bb, W.__getitem__, np.asarray(seq))
    for l in range(bb["n_layers"]):
        h = O.layer_forward(bb, W.__getitem__, task, l, h)
    assert np.allclose(scores[3], W["lm_head.W"] @ O.rms_norm(h, W["final.g"], bb["norm_eps"])[-1], rtol=1e-12, atol=1e-12)
    no_adapter = dict(task, adapters={})
    assert np.abs(D.lm_scores(bb, W.__getitem__, no_adapter, seq) - scores[3]).max() > 1e-2


# ---------------------------------------------------------------- image patch embedding vs nn.Conv2d (the ViT formulation)
def test_image_patch_embedding_matches_conv2d_patchify():
    C, HW, P, d = 3, 28, 14, 20
    r = _rng(14)
    img = r.random((C, HW, HW))
    W = {"embed.W": r.standard_normal((d, C * P * P)) * 0.1, "embed.b": r.standard_normal(d) * 0.1,
         "embed.cls": r.standard_normal(d), "embed.pos": r.standard_normal(((HW // P) ** 2 + 1, d)) * 0.1}
    bb = dict(input_kind="patch", patch_dim=C * P * P, has_cls=True, has_pos=True, img_c=C, img_hw=HW, patch_hw=P)
    got = O.tokens_from_input(bb, W.__getitem__, img.reshape(-1))
    conv = torch.nn.Conv2d(C, d, kernel_size=P, stride=P, **T64)
    with torch.no_grad():
        conv.weight.copy_(_t(W["embed.W"]).view(d, C, P, P))       # a ViT patch embed IS this convolution
        conv.bias.copy_(_t(W["embed.b"]))
        tok = conv(_t(img)[None])[0].flatten(1).transpose(0, 1)      # [grid*grid, d], patches row-major over the grid
        ref = torch.cat([_t(W["embed.cls"])[None], tok]) + _t(W["embed.pos"])
    assert got.shape == (5, d) and np.allclose(got, ref.numpy(), rtol=1e-12, atol=1e-13)


# ---------------------------------------------------------------- MLP decoder head vs nn.Sequential
def test_mlp_head_matches_torch_sequential_and_reduces_to_the_linear_head():
    d, hidden, out, n = 24, 16, 3, 7
    r = _rng(128)
    W = {"final.g": 1 + 0.1 * r.standard_normal(d), "final.b": 0.1 * r.standard_normal(d),
         "task004.head.W": r.standard_normal((hidden, d)), "task004.head.b": r.standard_normal(hidden),
         "task004.head.W2": r.standard_normal((out, hidden)), "task004.head.b2": r.standard_normal(out)}
    bb = dict(norm="ln", norm_eps=1e-5)
    h = r.standard_normal((n, d))
    for kind in ("mean", "cls", "last"):
        task = dict(id=4, adapters={}, head_kind=kind, head_out=out, head_hidden=hidden)
        got = O.head_forward(bb, W.__getitem__, task, h)
        f = F.layer_norm(_t(h), (d,), _t(W["final.g"]), _t(W["final.b"]), 1e-5)
        feat = {"mean": f.mean(0), "cls": f[0], "last": f[-1]}[kind]
        mlp = torch.nn.Sequential(torch.nn.Linear(d, hidden, **T64), torch.nn.ReLU(), torch.nn.Linear(hidden, out, **T64))
        with torch.no_grad():
            mlp[0].weight.copy_(_t(W["task004.head.W"])); mlp[0].bias.copy_(_t(W["task004.head.b"]))
            mlp[2].weight.copy_(_t(W["task004.head.W2"])); mlp[2].bias.copy_(_t(W["task004.head.b2"]))
            ref = mlp(feat).numpy()
        assert got.shape == (out,) and np.allclose(got, ref, rtol=1e-12, atol=1e-12)
    # special case: identity second layer on a non-negative hidden vector gives the first layer back
    W["task004.head.W"] = np.abs(W["task004.head.W"]); W["task004.head.b"] = np.abs(W["task004.head.b"])
    W["task004.head.W2"] = np.eye(hidden); W["task004.head.b2"] = np.zeros(hidden)
    pos = dict(norm="rms", norm_eps=1e-6)
    hp = np.abs(h)
    W["final.g"] = np.abs(W["final.g"])
    lin = O.head_forward(pos, W.__getitem__, dict(id=4, adapters={}, head_kind="mean", head_out=hidden), hp)
    mlp_out = O.head_forward(pos, W.__getitem__, dict(id=4, adapters={}, head_kind="mean", head_out=hidden, head_hidden=hidden), hp)
    assert (lin > 0).all() and np.allclose(lin, mlp_out, rtol=1e-13)


def test_dense_head_is_a_1x1_convolution_over_tokens_and_reduces_to_the_last_token_head():
    """SURVEY.md 8(f) NEXT-1, dense decoders: the head applied to every token row.  Pinned against
    torch.nn.Conv1d(d, o, kernel_size=1) over the token axis (the standard segmentation-style linear decoder), against the
    per-token scalar evaluation, and against the special case that its last row IS the last-token head."""
    d, out, n = 24, 5, 9
    r = _rng(70)
    W = {"final.g": 1 + 0.1 * r.standard_normal(d), "final.b": 0.1 * r.standard_normal(d),
         "task002.head.W": r.standard_normal((out, d)), "task002.head.b": r.standard_normal(out)}
    bb = dict(norm="ln", norm_eps=1e-5)
    h = r.standard_normal((n, d))
    got = O.head_forward(bb, W.__getitem__, dict(id=2, adapters={}, head_kind="dense", head_out=out), h)
    assert got.shape == (n * out,)
    f = F.layer_norm(_t(h), (d,), _t(W["final.g"]), _t(W["final.b"]), 1e-5)
    conv = torch.nn.Conv1d(d, out, kernel_size=1, **T64)
    with torch.no_grad():
        conv.weight.copy_(_t(W["task002.head.W"])[:, :, None]); conv.bias.copy_(_t(W["task002.head.b"]))
        ref = conv(f.T[None])[0].T.numpy()                       # [n, out]
    assert np.allclose(got.reshape(n, out), ref, rtol=1e-12, atol=1e-12)
    fn = f.numpy()
    for tok in (0, 4, n - 1):
        for o in range(out):
            want = sum(W["task002.head.W"][o, c] * fn[tok, c] for c in range(d)) + W["task002.head.b"][o]
            assert abs(got[tok * out + o] - want) < 1e-12        # layout: token-major, then class
    last = O.head_forward(bb, W.__getitem__, dict(id=2, adapters={}, head_kind="last", head_out=out), h)
    assert np.allclose(got.reshape(n, out)[-1], last, rtol=1e-13, atol=1e-13)


# ---------------------------------------------------------------- per-task input encoder
def test_input_channel_combiner_is_a_1x1_convolution_and_reduces_to_the_plain_path():
    C, n_patches, pdim, d = 3, 6, 8, 12
    r = _rng(31)
    W = {"embed.W": r.standard_normal((d, pdim)), "embed.b": r.standard_normal(d), "embed.pos": r.standard_normal((n_patches, d)),
         "task002.enc.W": r.standard_normal(C), "task002.enc.b": r.standard_normal(1)}
    bb = dict(input_kind="patch", patch_dim=pdim, has_cls=False, has_pos=True, img_c=0, img_hw=0, patch_hw=0)
    task = dict(id=2, adapters={}, head_kind="mean", head_out=1, enc_channels=C)
    x = r.standard_normal((C, n_patches * pdim))
    got = O.tokens_from_input(bb, W.__getitem__, x.reshape(-1), task)
    conv = torch.nn.Conv1d(C, 1, kernel_size=1, **T64)              # LinearChannelCombiner(C -> 1) is a 1x1 convolution
    with torch.no_grad():
        conv.weight.copy_(_t(W["task002.enc.W"]).view(1, C, 1)); conv.bias.copy_(_t(W["task002.enc.b"]))
        series = conv(_t(x)[None])[0, 0].numpy()
    ref = O.tokens_from_input(bb, W.__getitem__, series)             # the plain single-channel path on the combined series
    assert got.shape == (n_patches, d) and np.allclose(got, ref, rtol=1e-12, atol=1e-12)
    # one-hot weights, zero bias: the encoder picks a channel
    W["task002.enc.W"] = np.array([0.0, 1.0, 0.0]); W["task002.enc.b"] = np.zeros(1)
    assert np.allclose(O.tokens_from_input(bb, W.__getitem__, x.reshape(-1), task), O.tokens_from_input(bb, W.__getitem__, x[1]))


# ---------------------------------------------------------------- NEXT-4 variant: T5 relative-position bias vs transformers' T5
def test_relative_position_bucket_matches_hf_t5():
    tr = pytest.importorskip("transformers")
    from transformers.models.t5.modeling_t5 import T5Attention
    rel = torch.arange(-400, 401, dtype=torch.long)
    for bidirectional in (True, False):
        for n_buckets, max_distance in ((32, 128), (8, 20), (16, 64), (32, 1024)):
            want = T5Attention._relative_position_bucket(rel, bidirectional=bidirectional, num_buckets=n_buckets, max_distance=max_distance)
            got = [O.rel_bucket(int(x), bidirectional, n_buckets, max_distance) for x in rel]
            assert got == want.tolist(), (bidirectional, n_buckets, max_distance)


def test_t5_encoder_block_with_relative_bias_matches_hf_t5block():
    """cfg2's family (RMSNorm, ReLU, no biases) + the relative-position bias = a T5 encoder block.  T5 does not scale the scores
    by 1/sqrt(d_h) (SURVEY.md 8(c) reading 1 keeps the scale), so the HF block gets Wq / sqrt(d_h): sqrt(16) = 4, exact."""
    tr = pytest.importorskip("transformers")
    from transformers.models.t5.modeling_t5 import T5Block
    d, H, dh, Fd, n, NB, MD = 64, 4, 16, 96, 45, 8, 20                  # n > max distance: the last bucket is exercised
    cfg = tr.T5Config(d_model=d, d_kv=dh, num_heads=H, d_ff=Fd, num_layers=1, relative_attention_num_buckets=NB,
                      relative_attention_max_distance=MD, dropout_rate=0.0, layer_norm_epsilon=1e-6, feed_forward_proj="relu",
                      is_decoder=False, use_cache=False)
    cfg._attn_implementation = "eager"
    r = _rng(77)
    W = {"rel_bias.W": r.standard_normal((NB, H))}
    p = "L00."
    for nm, shape in (("Wq", (d, d)), ("Wk", (d, d)), ("Wv", (d, d)), ("Wo", (d, d)), ("Wup", (Fd, d)), ("Wdown", (d, Fd))):
        W[p + nm] = r.standard_normal(shape) * 0.2
    for nm in ("norm1", "norm2"):
        W[p + nm + ".g"] = 1 + 0.1 * r.standard_normal(d)
    bb = dict(n_layers=1, d_model=d, n_q_heads=H, n_kv_heads=H, head_dim=dh, d_ffn=Fd, act="relu", norm="rms", norm_eps=1e-6,
              causal=False, rope_theta=0.0, input_kind="embedded", patch_dim=0, has_cls=False, has_bias=False, has_pos=False,
              img_c=0, img_hw=0, patch_hw=0, rel_buckets=NB, rel_max_distance=MD)
    x = r.standard_normal((n, d))
    got = O.layer_forward(bb, W.__getitem__, None, 0, x)
    # without the bias the result must differ (the pin would not see a dropped term otherwise)
    assert np.abs(got - O.layer_forward({**bb, "rel_buckets": 0}, W.__getitem__, None, 0, x)).max() > 1e-3

    blk = T5Block(cfg, has_relative_attention_bias=True, layer_idx=0).to(torch.float64).eval()
    with torch.no_grad():
        sa = blk.layer[0].SelfAttention
        sa.q.weight.copy_(_t(W[p + "Wq"] / math.sqrt(dh)))
        sa.k.weight.copy_(_t(W[p + "Wk"]))
        sa.v.weight.copy_(_t(W[p + "Wv"]))
        sa.o.weight.copy_(_t(W[p + "Wo"]))
        sa.relative_attention_bias.weight.copy_(_t(W["rel_bias.W"]))
        blk.layer[0].layer_norm.weight.copy_(_t(W[p + "norm1.g"]))
        ff = blk.layer[1]
        ff.DenseReluDense.wi.weight.copy_(_t(W[p + "Wup"]))
        ff.DenseReluDense.wo.weight.copy_(_t(W[p + "Wdown"]))
        ff.layer_norm.weight.copy_(_t(W[p + "norm2.g"]))
        try:
            out = blk(_t(x)[None], cache_position=torch.arange(n))
        except TypeError:
            out = blk(_t(x)[None])
    want = (out[0] if isinstance(out, (tuple, list)) else out)[0].numpy()
    # HF's T5 takes the softmax and the RMS statistics in float32 whatever the module's dtype (`scores.float()`), so the two agree
    # to float32 rounding of O(1) values, not to 1e-10; a wrong bucket or a dropped bias is > 1e-3 (asserted above)
    assert np.allclose(got, want, rtol=0, atol=2e-5), np.abs(got - want).max()
