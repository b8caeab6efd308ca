"""Algorithmic work of one mixed-task forward.

Counts ONLY what the method itself must compute or move: no padding rows, no zero-padded rank
columns, no masked upper triangle.  Used by bench.py for "% of tensor peak" and the roofline.
Pure arithmetic on shapes; nothing here touches a tensor.
"""
from fmx_workloads import Workload, target_dims


def flops(wl: Workload) -> dict:
    """-> dict of algorithmic FLOPs per forward, by component, plus 'total' and the per-GEMM-family
    split {'gemm_qkv','gemm_o','gemm_ffn_in','gemm_ffn_out'} (base projection + fused LoRA expand)."""
    bb = wl.bb
    L, d, dq, dkv, F = bb.n_layers, bb.d_model, bb.d_q, bb.d_kv, bb.d_ffn
    N = wl.n_tokens
    k_in = 2 if bb.act == "swiglu" else 1
    fam = {
        "gemm_qkv": 2.0 * N * d * (dq + 2 * dkv) * L,
        "gemm_o": 2.0 * N * dq * d * L,
        "gemm_ffn_in": 2.0 * N * d * F * k_in * L,
        "gemm_ffn_out": 2.0 * N * F * d * L,
    }
    base = sum(fam.values())
    fam_of = {"q": "gemm_qkv", "k": "gemm_qkv", "v": "gemm_qkv", "o": "gemm_o", "gate": "gemm_ffn_in",
              "up": "gemm_ffn_in", "down": "gemm_ffn_out"}
    shrink = expand = 0.0
    shrink_fam = {k: 0.0 for k in fam}          # shrink FLOPs by the GEMM family that consumes (and, when fused, computes) them
    for t, n in zip(wl.task_ids, wl.lengths):
        for ad in wl.tasks[int(t)].adapters:
            din, dout = target_dims(bb, ad.target)
            sh = 2.0 * int(n) * ad.rank * din * L
            shrink += sh
            shrink_fam[fam_of[ad.target]] += sh
            e = 2.0 * int(n) * ad.rank * dout * L
            expand += e
            fam[fam_of[ad.target]] += e
    attn = 0.0
    for n in wl.lengths:
        n = int(n)
        attn += 4.0 * bb.n_q_heads * bb.head_dim * (n * (n + 1) / 2 if bb.causal else n * n) * L
    head = sum(2.0 * wl.tasks[int(t)].d_feat(bb) * wl.tasks[int(t)].head_out for t in wl.task_ids)
    embed = 2.0 * bb.patch_dim * d * bb.n_patches * wl.n_req if bb.input_kind == "patch" else 0.0
    total = base + shrink + expand + attn + head + embed
    return dict(base_gemm=base, lora_shrink=shrink, lora_expand=expand, attention=attn, head=head, embed=embed,
                total=total, families=fam, shrink_families=shrink_fam)


def gemm_launches_per_forward(wl: Workload) -> int:
    return 4 * wl.bb.n_layers


def norm_bytes_per_launch(wl: Workload) -> float:
    """S3a: fp32 read + bf16 write per element."""
    return wl.n_tokens * wl.bb.d_model * 6.0
