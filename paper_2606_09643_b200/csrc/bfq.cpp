// BFQ — batch-aware fair-queue batch builder (host only, no CUDA).
// PAPER.md §4.2: Eq. 1 (L156) S = max{F_prev, v}; Eq. 2 (L158) F = S + l/w; v = max_i F_i^last
// over each task's most recently dispatched request (L160); batch formation by start tag until
// B_max or an SLO violation (L160); Eq. 3 (L164) retag with l_i(b); token-level charging (L168).
// Readings of the open points: DESIGN.md §3 (24-29).  All tag arithmetic is IEEE double in the
// order written; compiled with -ffp-contract=off.
#include <algorithm>
#include <cmath>
#include <deque>
#include <new>
#include <vector>

#include "fmx.h"
#include "common.h"

namespace {
struct Req {
  int32_t task;
  uint64_t handle;
  int32_t n;
  double arrival, S, F, v_arr;
  uint64_t seq;
};
}  // namespace

struct fmx_bfq {
  int32_t n_tasks, b_max;
  std::vector<double> lat;
  double l_tok;
  std::vector<double> w, slo, F_prev, F_last, F_base, service_ms;
  std::vector<int64_t> dispatched;
  std::vector<std::deque<Req>> queue;
  std::vector<Req> last_batch;
  uint64_t seq = 0;

  double l_single(int32_t n) const { return l_tok > 0.0 ? l_tok * n : lat[0]; }
  double lat_batch(int32_t b, int64_t tokens) const { return l_tok > 0.0 ? l_tok * (double)tokens : lat[b - 1]; }
};

extern "C" {

int fmx_bfq_create(const fmx_bfq_params *p, fmx_bfq **out) {
  if (!p || !out || !p->lat_ms) return fmx_fail(FMX_E_INVALID_ARG, "bfq_create: NULL argument");
  if (p->n_tasks < 1 || p->n_tasks > FMX_MAX_TASKS || p->b_max < 1)
    return fmx_fail(FMX_E_INVALID_ARG, "bfq_create: n_tasks in [1,%d], b_max >= 1", FMX_MAX_TASKS);
  fmx_bfq *q = new (std::nothrow) fmx_bfq();
  if (!q) return fmx_fail(FMX_E_CAPACITY, "bfq_create: out of memory");
  q->n_tasks = p->n_tasks;
  q->b_max = p->b_max;
  q->lat.assign(p->lat_ms, p->lat_ms + p->b_max);
  q->l_tok = p->l_tok_ms;
  q->w.assign(p->n_tasks, 1.0);
  q->slo.assign(p->n_tasks, INFINITY);
  q->F_prev.assign(p->n_tasks, 0.0);
  q->F_last.assign(p->n_tasks, 0.0);
  q->F_base.assign(p->n_tasks, 0.0);
  q->service_ms.assign(p->n_tasks, 0.0);
  q->dispatched.assign(p->n_tasks, 0);
  q->queue.resize(p->n_tasks);
  *out = q;
  return FMX_OK;
}

int fmx_bfq_destroy(fmx_bfq *q) {
  delete q;
  return FMX_OK;
}

static int check_task(const fmx_bfq *q, fmx_task_t t, const char *who) {
  if (!q) return fmx_fail(FMX_E_INVALID_ARG, "%s: NULL queue", who);
  if (t < 0 || t >= q->n_tasks) return fmx_fail(FMX_E_UNKNOWN_TASK, "%s: task %d out of range", who, t);
  return FMX_OK;
}

int fmx_bfq_set_task(fmx_bfq *q, fmx_task_t task, double weight, double slo_ms) {
  if (int e = check_task(q, task, "bfq_set_task")) return e;
  if (!(weight > 0.0)) return fmx_fail(FMX_E_INVALID_ARG, "bfq_set_task: weight must be > 0");
  q->w[task] = weight;
  q->slo[task] = slo_ms;
  return FMX_OK;
}

int fmx_bfq_enqueue(fmx_bfq *q, fmx_task_t task, uint64_t req_handle, int32_t length, double arrival_ms) {
  if (int e = check_task(q, task, "bfq_enqueue")) return e;
  if (length < 1) return fmx_fail(FMX_E_BAD_LENGTH, "bfq_enqueue: length %d < 1", length);
  double v = q->F_last[0];
  for (int i = 1; i < q->n_tasks; ++i) v = std::max(v, q->F_last[i]);
  Req r;
  r.task = task; r.handle = req_handle; r.n = length; r.arrival = arrival_ms; r.v_arr = v;
  r.S = std::max(q->F_prev[task], v);                    // Eq. 1
  r.F = r.S + q->l_single(length) / q->w[task];          // Eq. 2
  r.seq = q->seq++;
  q->queue[task].push_back(r);
  q->F_prev[task] = r.F;
  return FMX_OK;
}

int fmx_bfq_next_batch(fmx_bfq *q, double now_ms, int32_t cap, int32_t *task_ids, int32_t *lengths,
                       uint64_t *req_handles, int32_t *n_out) {
  if (!q || !n_out) return fmx_fail(FMX_E_INVALID_ARG, "bfq_next_batch: NULL argument");
  std::vector<size_t> heads(q->n_tasks, 0);
  std::vector<Req> sel;
  int64_t tokens = 0;
  const int32_t limit = std::min(q->b_max, cap);
  for (;;) {
    const Req *best = nullptr;
    for (int i = 0; i < q->n_tasks; ++i) {               // k-way merge of the queue heads
      if (heads[i] >= q->queue[i].size()) continue;
      const Req *r = &q->queue[i][heads[i]];
      if (!best || r->S < best->S || (r->S == best->S && (r->F < best->F || (r->F == best->F && r->seq < best->seq))))
        best = r;
    }
    if (!best) break;
    const int32_t b = (int32_t)sel.size();
    if (b >= 1) {
      if (b + 1 > limit) break;
      const double done = now_ms + q->lat_batch(b + 1, tokens + best->n);
      bool late = done > best->arrival + q->slo[best->task];
      for (const Req &r : sel) late = late || (done > r.arrival + q->slo[r.task]);
      if (late) break;
    } else if (limit < 1) {
      break;
    }
    sel.push_back(*best);
    tokens += best->n;
    heads[best->task]++;
  }
  q->F_base = q->F_last;
  for (size_t j = 0; j < sel.size(); ++j) {
    const Req &r = sel[j];
    q->queue[r.task].pop_front();
    q->F_last[r.task] = r.F;
    q->dispatched[r.task]++;
    if (task_ids) task_ids[j] = r.task;
    if (lengths) lengths[j] = r.n;
    if (req_handles) req_handles[j] = r.handle;
  }
  q->last_batch = sel;
  *n_out = (int32_t)sel.size();
  return FMX_OK;
}

int fmx_bfq_complete(fmx_bfq *q, double measured_batch_ms) {
  if (!q) return fmx_fail(FMX_E_INVALID_ARG, "bfq_complete: NULL queue");
  std::vector<Req> &batch = q->last_batch;
  if (batch.empty()) return FMX_OK;
  const int32_t b_total = (int32_t)batch.size();
  int64_t tokens = 0;
  for (const Req &r : batch) tokens += r.n;
  const double total = measured_batch_ms > 0.0 ? measured_batch_ms : q->lat_batch(b_total, tokens);
  const bool tok = q->l_tok > 0.0;
  const double unit = tok ? total / (double)tokens : total / (double)b_total;
  auto l_b = [&](const Req &r) { return tok ? unit * r.n : unit; };   // l_i(b), Eq. 3
  std::vector<char> seen(q->n_tasks, 0);
  for (const Req &r : batch) seen[r.task] = 1;
  for (int i = 0; i < q->n_tasks; ++i) {
    if (!seen[i]) continue;
    double F = q->F_base[i];
    for (Req &r : batch) {
      if (r.task != i) continue;
      r.S = std::max(F, r.v_arr);
      r.F = r.S + l_b(r) / q->w[i];
      F = r.F;
      q->service_ms[i] += l_b(r);
    }
    q->F_last[i] = F;
    for (Req &r : q->queue[i]) {
      r.S = std::max(F, r.v_arr);
      r.F = r.S + l_b(r) / q->w[i];
      F = r.F;
    }
    q->F_prev[i] = F;
  }
  batch.clear();
  return FMX_OK;
}

int fmx_bfq_stats(fmx_bfq *q, fmx_task_t task, int64_t *dispatched, double *service_ms, int32_t *queued) {
  if (int e = check_task(q, task, "bfq_stats")) return e;
  if (dispatched) *dispatched = q->dispatched[task];
  if (service_ms) *service_ms = q->service_ms[task];
  if (queued) *queued = (int32_t)q->queue[task].size();
  return FMX_OK;
}

int fmx_bfq_peek(fmx_bfq *q, fmx_task_t task, int32_t j, double *out3) {
  if (int e = check_task(q, task, "bfq_peek")) return e;
  if (!out3 || j < 0 || (size_t)j >= q->queue[task].size()) return fmx_fail(FMX_E_INVALID_ARG, "bfq_peek: bad index");
  const Req &r = q->queue[task][j];
  out3[0] = r.S; out3[1] = r.F; out3[2] = r.v_arr;
  return FMX_OK;
}

}  // extern "C"
