"""Session: upload a seeded `fmx_workloads.Workload` to the GPU and run it through libfmx.

Marshalling only — torch provides device memory and streams; every compute step is in libfmx.
"""
import time

import numpy as np
import torch

from fmx_workloads import Workload, target_dims
from .binding import ACT, HEAD_KIND, INPUT_KIND, NORM, TARGET, Fmx


def _dev_bf16(bits, device):
    """uint16 bf16 bit patterns -> torch.bfloat16 tensor on the device (same bits)."""
    t = torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).to(device)
    return t.view(torch.bfloat16)


class Session:
    def __init__(self, wl: Workload, device=0, fmx: Fmx = None, max_req=None, max_tokens=None, weights_from=None):
        """weights_from: another Session on a backbone of the SAME shape whose device-resident backbone tensors are reused
        instead of generating and uploading this workload's own (timing runs that only change the task set: same shapes,
        same value distribution; never used by a parity test)."""
        self.wl = wl
        self.dev = torch.device("cuda", device)
        torch.cuda.set_device(self.dev)
        self.fmx = fmx or Fmx(device)
        self._weights = dict(weights_from._weights) if weights_from is not None else {}
        self.bb = self._register_backbone()
        self.task_ids_of = [self._register_task(t) for t in range(len(wl.tasks))]
        self.max_req = max_req or wl.n_req
        self.max_tokens = max_tokens or max(wl.n_tokens, 1)
        self._alloc_workspace(self.fmx.workspace_bytes(self.bb, self.max_req, self.max_tokens))
        self.inputs_dev = None
        self.out_dev = None

    def _alloc_workspace(self, nbytes):
        self.ws_bytes = nbytes
        self.workspace = torch.empty(nbytes + 1024, dtype=torch.uint8, device=self.dev)
        self.ws_ptr = (self.workspace.data_ptr() + 1023) // 1024 * 1024

    def ensure_host_workspace(self, input_bytes, output_floats):
        """fmx_forward_mixed_host stages the packed inputs and the outputs in the workspace too."""
        need = self.fmx.host_workspace_bytes(self.bb, self.max_req, self.max_tokens, input_bytes, output_floats)
        if need > self.ws_bytes:
            torch.cuda.synchronize(self.dev)
            self._alloc_workspace(need)

    # ------------------------------------------------------------------ registration
    def _w(self, name):
        if name not in self._weights:
            self._weights[name] = _dev_bf16(self.wl.tensor(name), self.dev)
        return self._weights[name].data_ptr()

    def _register_backbone(self):
        wl, bb = self.wl, self.wl.bb
        L = bb.n_layers
        fields = dict(n_layers=L, d_model=bb.d_model, n_q_heads=bb.n_q_heads, n_kv_heads=bb.n_kv_heads,
                      head_dim=bb.head_dim, d_ffn=bb.d_ffn, act=ACT[bb.act], norm=NORM[bb.norm], norm_eps=bb.norm_eps,
                      causal=int(bb.causal), rope_theta=bb.rope_theta, input_kind=INPUT_KIND[bb.input_kind],
                      patch_dim=bb.patch_dim, tokens_per_request=bb.tokens_per_request, has_cls=int(bb.has_cls),
                      vocab=bb.vocab, max_seq=bb.max_seq, img_c=bb.img_c, img_hw=bb.img_hw, patch_hw=bb.patch_hw,
                      rel_buckets=getattr(bb, "rel_buckets", 0), rel_max_distance=getattr(bb, "rel_max_distance", 0))
        lay = lambda n: [self._w(f"L{l:02d}.{n}") for l in range(L)]
        per_layer = dict(norm1_g=lay("norm1.g"), norm2_g=lay("norm2.g"), Wq=lay("Wq"), Wk=lay("Wk"), Wv=lay("Wv"),
                         Wo=lay("Wo"), Wup=lay("Wup"), Wdown=lay("Wdown"),
                         Wgate=lay("Wgate") if bb.act == "swiglu" else None,
                         norm1_b=lay("norm1.b") if bb.norm == "ln" else None,
                         norm2_b=lay("norm2.b") if bb.norm == "ln" else None)
        for b in ("bq", "bk", "bv", "bo", "bup", "bdown"):
            per_layer[b] = lay(b) if bb.has_bias else None
        per_layer["bgate"] = lay("bgate") if (bb.has_bias and bb.act == "swiglu") else None
        singles = dict(final_g=self._w("final.g"), final_b=self._w("final.b") if bb.norm == "ln" else None,
                       embed_W=self._w("embed.W") if bb.input_kind == "patch" else None,
                       embed_b=self._w("embed.b") if bb.input_kind == "patch" else None,
                       embed_cls=self._w("embed.cls") if bb.has_cls else None,
                       embed_pos=self._w("embed.pos") if bb.pos_kind != "none" else None,
                       embed_table=self._w("embed.table") if bb.input_kind == "tokens" else None,
                       rel_bias=self._w("rel_bias.W") if getattr(bb, "rel_buckets", 0) else None)
        return self.fmx.register_backbone(fields, per_layer, singles)

    def _register_task(self, t, presynced=None):
        wl, bb = self.wl, self.wl.bb
        ts = wl.tasks[t]
        tmp = []
        def up(name):
            if presynced is not None:                     # tensors uploaded (and synchronised) earlier
                return presynced[name].data_ptr()
            x = _dev_bf16(wl.tensor(name), self.dev)
            tmp.append(x)
            return x.data_ptr()
        adapters = []
        for ad in ts.adapters:
            A = [up(f"task{t:03d}.L{l:02d}.{ad.target}.A") for l in range(bb.n_layers)]
            Bm = [up(f"task{t:03d}.L{l:02d}.{ad.target}.B") for l in range(bb.n_layers)]
            adapters.append((TARGET[ad.target], ad.rank, float(ad.scaling), A, Bm))
        mlp = getattr(ts, "head_hidden", 0)
        enc = getattr(ts, "enc_channels", 0)
        head = (up(f"task{t:03d}.head.W"), up(f"task{t:03d}.head.b"))
        if presynced is None:
            torch.cuda.synchronize(self.dev)
        t0 = time.perf_counter()                         # the fmx_register_task call alone: tensors already on the device
        tid = self.fmx.register_task(self.bb, adapters, HEAD_KIND[ts.head_kind], ts.head_out,
                                     head[0], head[1], mlp,
                                     up(f"task{t:03d}.head.W2") if mlp else None, up(f"task{t:03d}.head.b2") if mlp else None,
                                     enc, up(f"task{t:03d}.enc.W") if enc > 1 else None, up(f"task{t:03d}.enc.b") if enc > 1 else None)
        self.last_register_ms = (time.perf_counter() - t0) * 1e3
        del tmp      # the library copied everything into its arena
        return tid

    def _register_task_presynced(self, t):
        """Upload workload task t's tensors, synchronise, and only then (when called) register: used to time the call while
        other work is queued on the device."""
        if not hasattr(self, "_pre"):
            self._pre = {}
        if t not in self._pre:
            names = self.wl.task_tensor_names(t)
            self._pre[t] = {n: _dev_bf16(self.wl.tensor(n), self.dev) for n in names}
            torch.cuda.synchronize(self.dev)
        return self._register_task(t, presynced=self._pre[t])

    def prepare_task_copy(self, t):
        """Upload (and synchronise) workload task t's tensors ahead of register_while_serving_ms."""
        if not hasattr(self, "_pre"):
            self._pre = {}
        names = self.wl.task_tensor_names(t)
        self._pre[t] = {n: _dev_bf16(self.wl.tensor(n), self.dev) for n in names}
        torch.cuda.synchronize(self.dev)

    def task_lifecycle_ms(self, t):
        """Unregister and re-register workload task t on the live context (R2 lifecycle decoupling): the
        backbone and every other task stay registered.  Returns (unregister_ms, register_ms) of the two C-ABI calls; the task
        keeps its slot (lowest free slot first), so the session's id map stays valid."""
        tid = self.task_ids_of[t]
        torch.cuda.synchronize(self.dev)
        t0 = time.perf_counter()
        self.fmx.unregister_task(tid)
        un_ms = (time.perf_counter() - t0) * 1e3
        new = self._register_task(t)
        assert new == tid, "a freed slot is reused lowest-first"
        return un_ms, self.last_register_ms

    def register_while_serving_ms(self, t, n_forwards=5, stream=None):
        """NEXT-2: add one more task (a copy of workload task t in a fresh slot) while `n_forwards` forwards
        are queued on the stream; returns (register_ms, forwards_ms, new task id).  fmx_register_task runs on the library's
        own stream and returns without waiting for the queued forwards."""
        s = stream if stream is not None else torch.cuda.current_stream(self.dev)
        if not hasattr(self, "_pre") or t not in self._pre:
            self.prepare_task_copy(t)
        self.forward(stream=s)
        s.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(s)
        for _ in range(n_forwards):
            self.forward(stream=s)
        e1.record(s)
        tid = self._register_task_presynced(t)
        reg_ms = self.last_register_ms
        s.synchronize()
        return reg_ms, e0.elapsed_time(e1), tid

    def unregister_while_serving_ms(self, t, n_forwards=5, stream=None):
        """NEXT-2: remove a fresh copy of workload task t (so the batch stays servable) while `n_forwards` forwards are queued; returns (unregister_ms, forwards_ms).  fmx_unregister_task does not
        synchronise the device: the copy's buffers are released on the device after the queued forwards."""
        s = stream if stream is not None else torch.cuda.current_stream(self.dev)
        tid = self._register_task_presynced(t)
        self.forward(stream=s)
        s.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(s)
        for _ in range(n_forwards):
            self.forward(stream=s)
        e1.record(s)
        t0 = time.perf_counter()
        self.fmx.unregister_task(tid)
        un_ms = (time.perf_counter() - t0) * 1e3
        s.synchronize()
        return un_ms, e0.elapsed_time(e1)

    # ------------------------------------------------------------------ token decode (NEXT-3)
    def enable_decode(self, n_slots, max_req=None):
        """Register the workload's LM head, allocate the KV cache for n_slots sequences and re-size the workspace (the LM
        scores buffer is part of it)."""
        self._lm = _dev_bf16(self.wl.tensor("lm_head.W"), self.dev)
        self.fmx.register_lm_head(self.bb, self._lm.data_ptr(), self.wl.bb.vocab)
        self.n_slots = n_slots
        self.kv_cache = torch.zeros(self.fmx.kv_cache_bytes(self.bb, n_slots) + 16, dtype=torch.uint8, device=self.dev)
        self.kv_ptr = (self.kv_cache.data_ptr() + 15) // 16 * 16
        if max_req:
            self.max_req = max_req
        self._alloc_workspace(self.fmx.workspace_bytes(self.bb, self.max_req, self.max_tokens))
        vocab = self.wl.bb.vocab
        self.scores_dev = torch.empty(self.max_req * vocab, dtype=torch.float32, device=self.dev)
        self.next_dev = torch.empty(self.max_req, dtype=torch.int32, device=self.dev)

    def prefill(self, tokens, task_ids, lengths, slots, with_heads=True, stream=None):
        """tokens: packed int32 prompts.  Returns (scores [B, vocab], next tokens [B], head outputs or None) as numpy."""
        ids = np.asarray([self.task_ids_of[int(t)] for t in task_ids], dtype=np.int32)
        B, vocab = len(ids), self.wl.bb.vocab
        tok = torch.from_numpy(np.ascontiguousarray(tokens, dtype=np.int32)).to(self.dev)
        out = None
        if with_heads:
            off = self.fmx.output_layout(ids)
            out = torch.empty(max(int(off[-1]), 1), dtype=torch.float32, device=self.dev)
        s = stream if stream is not None else torch.cuda.current_stream(self.dev)
        self.fmx.prefill(self.bb, tok.data_ptr(), ids, lengths, slots, out.data_ptr() if with_heads else 0, self.scores_dev.data_ptr(),
                         self.next_dev.data_ptr(), self.kv_ptr, self.n_slots, self.ws_ptr, self.ws_bytes, s.cuda_stream)
        torch.cuda.synchronize(self.dev)
        heads = None
        if with_heads:
            flat = out.cpu().numpy()
            heads = [flat[off[i]:off[i + 1]].copy() for i in range(B)]
        return self.scores_dev[:B * vocab].cpu().numpy().reshape(B, vocab), self.next_dev[:B].cpu().numpy(), heads

    def decode_step(self, tokens_dev_ptr, task_ids, slots, positions, want_scores=True, stream=None, sync=True):
        """One decode iteration; tokens_dev_ptr: device address of int32 [B].  Returns (scores or None, next tokens) as numpy
        when sync, else nothing (results stay in self.scores_dev / self.next_dev)."""
        ids = np.asarray([self.task_ids_of[int(t)] for t in task_ids], dtype=np.int32)
        B, vocab = len(ids), self.wl.bb.vocab
        s = stream if stream is not None else torch.cuda.current_stream(self.dev)
        self.fmx.decode_step(self.bb, tokens_dev_ptr, ids, slots, positions, self.scores_dev.data_ptr() if want_scores else 0,
                             self.next_dev.data_ptr(), self.kv_ptr, self.n_slots, self.ws_ptr, self.ws_bytes, s.cuda_stream)
        if not sync:
            return None
        torch.cuda.synchronize(self.dev)
        sc = self.scores_dev[:B * vocab].cpu().numpy().reshape(B, vocab) if want_scores else None
        return sc, self.next_dev[:B].cpu().numpy()

    # ------------------------------------------------------------------ running
    def upload_inputs(self, packed=None):
        packed = self.wl.packed_inputs() if packed is None else packed
        raw = np.ascontiguousarray(packed)
        self.inputs_host = torch.from_numpy(raw.view(np.int16) if raw.dtype == np.uint16 else raw).pin_memory()
        self.inputs_dev = self.inputs_host.to(self.dev)
        return self.inputs_dev

    def forward(self, task_ids=None, lengths=None, stream=None):
        """Enqueue one mixed forward on the current (or given) stream; returns the device output tensor."""
        wl = self.wl
        ids = wl.task_ids if task_ids is None else task_ids
        ids = np.asarray([self.task_ids_of[int(t)] for t in ids], dtype=np.int32)
        lens = wl.lengths if lengths is None else lengths
        if self.inputs_dev is None:
            self.upload_inputs()
        off = self.fmx.output_layout(ids, lens)
        if self.out_dev is None or self.out_dev.numel() < int(off[-1]):
            self.out_dev = torch.empty(max(int(off[-1]), 1), dtype=torch.float32, device=self.dev)
        s = stream if stream is not None else torch.cuda.current_stream(self.dev)
        self.fmx.forward_mixed(self.bb, self.inputs_dev.data_ptr(), ids, lens, self.out_dev.data_ptr(), self.ws_ptr,
                               self.ws_bytes, s.cuda_stream)
        self.last_off = off
        return self.out_dev

    def forward_numpy(self, task_ids=None, lengths=None):
        """Run and return a list of per-request fp32 output vectors (original request order)."""
        out = self.forward(task_ids, lengths)
        torch.cuda.synchronize(self.dev)
        flat = out.cpu().numpy()
        return [flat[self.last_off[i]:self.last_off[i + 1]].copy() for i in range(len(self.last_off) - 1)]
