// hpsi_stream_*: H psi with the operator arenas in pinned HOST memory, streamed through two device staging windows
// (SURVEY.md 8(f)-3).  The paper's runs leave HBM at D ~ 8-10k and become bound by host-device traffic
// ("host-device datacommunication ... due to memory limitations", "including host-device
// communication"); this entry point is that regime on one B200: the term list is cut into windows of terms whose
// blocks fit a staging buffer, every window gets its own plan bound to one of the two staging slots, and an apply
// copies window w+1 on a copy stream while window w computes; the windows' results add up in window order inside the
// ordered reduce (no atomics, bitwise reproducible).
#include <algorithm>
#include <cstdio>
#include <new>
#include <vector>

#include "plan_dev.h"

using namespace hpsi;

struct hpsi_stream {
  struct Window {
    hpsi_plan_t* plan = nullptr;
    int64_t a_lo = 0, a_len = 0, b_lo = 0, b_len = 0;   // host arena ranges (doubles) this window needs
  };
  std::vector<Window> win;
  const double* a_host = nullptr;
  const double* b_host = nullptr;
  double* stage[2] = {nullptr, nullptr};                // slot = [A window | B window]
  int64_t a_cap = 0, b_cap = 0;
  cudaStream_t copy = nullptr;
  cudaEvent_t ready[2] = {nullptr, nullptr}, freed[2] = {nullptr, nullptr};
  int64_t psi_len = 0, useful_flops = 0, bytes_per_apply = 0;
};

extern "C" void hpsi_stream_destroy(hpsi_stream_t* s) {
  if (!s) return;
  for (auto& w : s->win) hpsi_destroy(w.plan);
  for (int i = 0; i < 2; ++i) {
    cudaFree(s->stage[i]);
    if (s->ready[i]) cudaEventDestroy(s->ready[i]);
    if (s->freed[i]) cudaEventDestroy(s->freed[i]);
  }
  if (s->copy) cudaStreamDestroy(s->copy);
  cudaGetLastError();
  delete s;
}

extern "C" int hpsi_stream_create(const hpsi_sectors_t* sectors, const hpsi_terms_t* terms, int64_t window_doubles,
                                  uint32_t flags, hpsi_stream_t** out) {
  if (!sectors || !terms || !out) { set_error("null argument"); return HPSI_EINVAL; }
  *out = nullptr;
  if (flags & HPSI_PLAN_HOST_ONLY) { set_error("a streamed plan needs a device"); return HPSI_EINVAL; }
  if (!terms->a_data || !terms->b_data) { set_error("hpsi_stream_create needs the HOST arenas"); return HPSI_EINVAL; }
  if (window_doubles < 2) { set_error("window too small"); return HPSI_EINVAL; }
  const int T = terms->n_terms;
  // arena range of every term (its blocks need not be contiguous; the range is what gets copied)
  struct Range { int64_t a_lo, a_hi, b_lo, b_hi; };
  std::vector<Range> rg(T, Range{INT64_MAX, 0, INT64_MAX, 0});
  auto extent = [&](const hpsi_opblock_t& e, const int32_t* d, int nsec, bool tr) -> int64_t {
    if (e.row < 0 || e.row >= nsec || e.col < 0 || e.col >= nsec) return -1;
    const int64_t srows = tr ? d[e.col] : d[e.row], scols = tr ? d[e.row] : d[e.col];     // a transposed block stores d[col] x d[row]
    return e.offset + (srows - 1) * e.ld + scols;
  };
  for (int64_t i = 0; i < terms->n_a; ++i) {
    const hpsi_opblock_t& e = terms->a_blocks[i];
    const int64_t hi = extent(e, sectors->d_left, sectors->n_left, terms->a_transposed && terms->a_transposed[i]);
    if (e.term < 0 || e.term >= T || hi < 0 || e.offset < 0) { set_error("bad A block descriptor"); return HPSI_EINVAL; }
    rg[e.term].a_lo = std::min(rg[e.term].a_lo, e.offset & ~(int64_t)3);      // keep 32-byte alignment of the rows
    rg[e.term].a_hi = std::max(rg[e.term].a_hi, hi);
  }
  for (int64_t i = 0; i < terms->n_b; ++i) {
    const hpsi_opblock_t& e = terms->b_blocks[i];
    const int64_t hi = extent(e, sectors->d_right, sectors->n_right, terms->b_transposed && terms->b_transposed[i]);
    if (e.term < 0 || e.term >= T || hi < 0 || e.offset < 0) { set_error("bad B block descriptor"); return HPSI_EINVAL; }
    rg[e.term].b_lo = std::min(rg[e.term].b_lo, e.offset & ~(int64_t)3);
    rg[e.term].b_hi = std::max(rg[e.term].b_hi, hi);
  }
  hpsi_stream_t* s = new (std::nothrow) hpsi_stream_t();
  if (!s) { set_error("out of host memory"); return HPSI_ENOMEM; }
  s->a_host = terms->a_data;
  s->b_host = terms->b_data;
  // windows of terms whose A + B ranges fit window_doubles.  The terms are taken in the order of their arena position
  // (ties: term number), so that terms which share storage - an adjoint reading its partner's blocks transposed - fall
  // into the same window and their bytes cross the host link once.  `order[cuts[w].first .. cuts[w].second)` = window w.
  std::vector<int> order(T);
  for (int t = 0; t < T; ++t) order[t] = t;
  std::stable_sort(order.begin(), order.end(), [&](int x, int y) {
    if (rg[x].a_lo != rg[y].a_lo) return rg[x].a_lo < rg[y].a_lo;
    return rg[x].b_lo < rg[y].b_lo;
  });
  std::vector<std::pair<int, int>> cuts;
  {
    int t0 = 0;
    Range cur{INT64_MAX, 0, INT64_MAX, 0};
    auto size = [](const Range& r) { return std::max<int64_t>(0, r.a_hi - std::min(r.a_lo, r.a_hi)) + std::max<int64_t>(0, r.b_hi - std::min(r.b_lo, r.b_hi)); };
    for (int i = 0; i < T; ++i) {
      const Range& rt = rg[order[i]];
      Range nx{std::min(cur.a_lo, rt.a_lo), std::max(cur.a_hi, rt.a_hi), std::min(cur.b_lo, rt.b_lo), std::max(cur.b_hi, rt.b_hi)};
      if (size(nx) > window_doubles && i > t0) {
        cuts.push_back({t0, i});
        t0 = i;
        nx = rt;
      }
      if (size(nx) > window_doubles) { set_error("one term's blocks do not fit the window"); hpsi_stream_destroy(s); return HPSI_EINVAL; }
      cur = nx;
    }
    if (T > t0 || T == 0) cuts.push_back({t0, T});
  }
  std::vector<int> window_of(T, 0);
  for (size_t w = 0; w < cuts.size(); ++w)
    for (int i = cuts[w].first; i < cuts[w].second; ++i) window_of[order[i]] = (int)w;
  int rc = HPSI_OK;
  auto fail = [&](int code) { hpsi_stream_destroy(s); return code; };
  // staging capacity = the largest window of each side
  std::vector<Range> wr(cuts.size(), Range{INT64_MAX, 0, INT64_MAX, 0});
  for (size_t w = 0; w < cuts.size(); ++w)
    for (int i = cuts[w].first; i < cuts[w].second; ++i) {
      const int t = order[i];
      wr[w].a_lo = std::min(wr[w].a_lo, rg[t].a_lo); wr[w].a_hi = std::max(wr[w].a_hi, rg[t].a_hi);
      wr[w].b_lo = std::min(wr[w].b_lo, rg[t].b_lo); wr[w].b_hi = std::max(wr[w].b_hi, rg[t].b_hi);
    }
  for (auto& r : wr) {
    if (r.a_lo > r.a_hi) r.a_lo = r.a_hi = 0;
    if (r.b_lo > r.b_hi) r.b_lo = r.b_hi = 0;
    s->a_cap = std::max(s->a_cap, (r.a_hi - r.a_lo + 3) & ~(int64_t)3);
    s->b_cap = std::max(s->b_cap, r.b_hi - r.b_lo);
  }
  for (int i = 0; i < 2; ++i) {
    if (cudaMalloc(&s->stage[i], std::max<int64_t>(s->a_cap + s->b_cap, 4) * sizeof(double)) != cudaSuccess) {
      cudaGetLastError();
      set_error("staging window allocation failed");
      return fail(HPSI_ENOMEM);
    }
    if (cudaEventCreateWithFlags(&s->ready[i], cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&s->freed[i], cudaEventDisableTiming) != cudaSuccess) return fail(cuda_fail(cudaGetLastError(), "cudaEventCreate"));
  }
  if (cudaStreamCreateWithFlags(&s->copy, cudaStreamNonBlocking) != cudaSuccess) return fail(cuda_fail(cudaGetLastError(), "cudaStreamCreate"));
  // one plan per window: only that window's blocks, offsets rebased to the staging slot
  for (size_t w = 0; w < cuts.size(); ++w) {
    std::vector<hpsi_opblock_t> ab, bb;
    std::vector<uint8_t> atr, btr;
    for (int64_t i = 0; i < terms->n_a; ++i)
      if (window_of[terms->a_blocks[i].term] == (int)w) {
        ab.push_back(terms->a_blocks[i]);
        ab.back().offset -= wr[w].a_lo;
        atr.push_back(terms->a_transposed ? terms->a_transposed[i] : 0);
      }
    for (int64_t i = 0; i < terms->n_b; ++i)
      if (window_of[terms->b_blocks[i].term] == (int)w) {
        bb.push_back(terms->b_blocks[i]);
        bb.back().offset -= wr[w].b_lo;
        btr.push_back(terms->b_transposed ? terms->b_transposed[i] : 0);
      }
    hpsi_terms_t sub = *terms;
    sub.n_a = (int64_t)ab.size(); sub.a_blocks = ab.data();
    sub.n_b = (int64_t)bb.size(); sub.b_blocks = bb.data();
    sub.a_transposed = terms->a_transposed ? atr.data() : nullptr;
    sub.b_transposed = terms->b_transposed ? btr.data() : nullptr;
    double* slot = s->stage[w & 1];
    sub.a_data = slot; sub.b_data = slot + s->a_cap;
    sub.a_len = s->a_cap; sub.b_len = s->b_cap;
    hpsi_stream::Window win;
    win.a_lo = wr[w].a_lo; win.a_len = wr[w].a_hi - wr[w].a_lo;
    win.b_lo = wr[w].b_lo; win.b_len = wr[w].b_hi - wr[w].b_lo;
    if ((rc = hpsi_plan(sectors, &sub, flags, &win.plan)) != HPSI_OK) return fail(rc);
    s->win.push_back(win);
    int64_t v = 0;
    hpsi_query(win.plan, HPSI_Q_USEFUL_FLOPS, &v, sizeof v); s->useful_flops += v;
    hpsi_query(win.plan, HPSI_Q_PSI_LENGTH, &v, sizeof v); s->psi_len = v;
    s->bytes_per_apply += 8 * (win.a_len + win.b_len);
  }
  *out = s;
  return HPSI_OK;
}

extern "C" int hpsi_stream_apply(hpsi_stream_t* s, const double* psi_dev, double* out_dev, void* cuda_stream) {
  if (!s || !psi_dev || !out_dev) { set_error("null argument"); return HPSI_EINVAL; }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (s->win.empty() || s->psi_len == 0) return HPSI_OK;
  for (size_t w = 0; w < s->win.size(); ++w) {
    const hpsi_stream::Window& win = s->win[w];
    const int slot = (int)(w & 1);
    HPSI_CUDA(cudaStreamWaitEvent(s->copy, s->freed[slot], 0));          // the window that used this slot has computed
    if (win.a_len > 0)
      HPSI_CUDA(cudaMemcpyAsync(s->stage[slot], s->a_host + win.a_lo, win.a_len * sizeof(double), cudaMemcpyHostToDevice, s->copy));
    if (win.b_len > 0)
      HPSI_CUDA(cudaMemcpyAsync(s->stage[slot] + s->a_cap, s->b_host + win.b_lo, win.b_len * sizeof(double), cudaMemcpyHostToDevice, s->copy));
    HPSI_CUDA(cudaEventRecord(s->ready[slot], s->copy));
    HPSI_CUDA(cudaStreamWaitEvent(st, s->ready[slot], 0));
    int rc = apply_impl(win.plan, psi_dev, out_dev, w > 0, cuda_stream);
    if (rc != HPSI_OK) return rc;
    HPSI_CUDA(cudaEventRecord(s->freed[slot], st));
  }
  return HPSI_OK;
}

extern "C" int hpsi_stream_query(const hpsi_stream_t* s, int what, void* out, size_t bytes) {
  if (!s || !out || bytes < sizeof(int64_t)) { set_error("bad argument"); return HPSI_EINVAL; }
  int64_t v;
  switch (what) {
    case HPSI_Q_PSI_LENGTH: v = s->psi_len; break;
    case HPSI_Q_USEFUL_FLOPS: v = s->useful_flops; break;
    case HPSI_Q_OPERATOR_BYTES: v = s->bytes_per_apply; break;          // bytes copied host -> device per apply
    case HPSI_SQ_N_WINDOWS: v = (int64_t)s->win.size(); break;
    case HPSI_SQ_STAGING_BYTES: v = 2 * (s->a_cap + s->b_cap) * (int64_t)sizeof(double); break;
    default: set_error("unknown stream query"); return HPSI_EINVAL;
  }
  *static_cast<int64_t*>(out) = v;
  return HPSI_OK;
}
