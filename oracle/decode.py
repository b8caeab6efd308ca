"""ORACLE (test infrastructure) — token decode of a mixed-task batch.

The paper serves "token-based FMs (e.g., LLMs with continuous batching and long-lived decode
iterations)" through the same vFM boundary (§4.2, fourth difference) and charges
"token-level work in service-time units" (L168); its prototype maps the boundary onto vLLM (L253).
It gives no arithmetic for a decode iteration, so the oracle is the plain definition:

    the next-token scores of request i, which has seen the tokens x_0 .. x_{n-1} and belongs to
    task t, are  LMHead( FinalNorm( Backbone_t(x_0 .. x_{n-1}) )[n-1] ),

i.e. the LAST row of the ordinary causal forward over the whole prefix with task t's adapters
(`oracle.vfm_forward`, step 1-3), times the language-model head matrix.  A key/value cache is an
implementation device that must not change this value: under a causal mask row n-1 of the full
forward depends on the earlier rows only through their keys and values, which are what a cache
stores.  The oracle therefore recomputes the whole prefix for every step - no cache, no batching,
fp64 - and greedy decoding appends argmax(scores).  (reading 34: the LM head is a
backbone-level matrix `lm_head.W` [vocab, d_model], not tied to the embedding table.)

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference legs may import this.
"""
import numpy as np

from .vfm_forward import _norm, layer_forward, tokens_from_input


def lm_scores(bb, get, task, tokens):
    """Next-token scores [vocab] after the prefix `tokens` (int array, length >= 1) for `task`."""
    tokens = np.asarray(tokens, dtype=np.int64)
    h = tokens_from_input(bb, get, tokens, task)
    for l in range(bb["n_layers"]):
        h = layer_forward(bb, get, task, l, h)
    f = _norm(bb, get, "final", h)
    return get("lm_head.W") @ f[-1]


def greedy_decode(bb, get, task, prompt, n_new, forced=None):
    """Decode `n_new` tokens after `prompt`.  Returns (tokens appended, list of score vectors).
    forced: optional sequence of tokens to append instead of the oracle's own argmax (teacher
    forcing: scores for the prefix ANOTHER implementation produced, so that a near-tie between
    the two best scores cannot make the sequences diverge)."""
    seq = [int(t) for t in prompt]
    out, scores = [], []
    for s in range(n_new):
        z = lm_scores(bb, get, task, seq)
        scores.append(z)
        nxt = int(forced[s]) if forced is not None else int(np.argmax(z))
        out.append(nxt)
        seq.append(nxt)
    return out, scores
