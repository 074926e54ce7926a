// C-ABI entry points of include/hpsi.h (plan / bind / apply / query / destroy / debug).
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include <cuda.h>

#include "plan_dev.h"

namespace hpsi {
static thread_local std::string g_err;
void set_error(const std::string& s) { g_err = s; }
int cuda_fail(cudaError_t e, const char* what) {
  g_err = std::string("CUDA error: ") + cudaGetErrorString(e) + " in " + what;
  cudaGetLastError();
  return HPSI_ECUDA;
}
}  // namespace hpsi

using namespace hpsi;

extern "C" const char* hpsi_last_error(void) { return g_err.c_str(); }

namespace hpsi {

template <class T>
static size_t table_bytes(const std::vector<T>& v) { return (v.size() * sizeof(T) + 255) / 256 * 256 + 256; }

template <class T>
static int upload(const std::vector<T>& v, char* base, size_t& cursor, const T** dev_ptr) {
  *dev_ptr = reinterpret_cast<const T*>(base + cursor);
  if (!v.empty()) HPSI_CUDA(cudaMemcpy(base + cursor, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice));
  cursor += table_bytes(v);
  return HPSI_OK;
}

int upload_schedule(hpsi_plan_t* p) {
  const Schedule& sc = p->sc;
  size_t total = table_bytes(sc.blocks) + table_bytes(sc.segs) + table_bytes(sc.groups) + table_bytes(sc.p1) +
                 table_bytes(sc.runs) + table_bytes(sc.p2) + table_bytes(sc.pf) + table_bytes(sc.diag) + table_bytes(sc.elem);
  HPSI_CUDA(cudaMalloc(&p->d_tables, total));
  cudaError_t e = cudaMalloc(&p->d_ws, (size_t)sc.ws_len * sizeof(double));
  if (e != cudaSuccess) {
    cudaGetLastError();
    char buf[160];
    snprintf(buf, sizeof buf, "device workspace allocation of %.2f GB failed", sc.ws_len * 8.0 / 1e9);
    set_error(buf);
    return HPSI_ENOMEM;
  }
  HPSI_CUDA(cudaMemset(p->d_ws, 0, (size_t)sc.ws_len * sizeof(double)));
  HPSI_CUDA(cudaMalloc(&p->d_maps, std::max<size_t>(sc.maps.size(), 1) * TMAP_BYTES));
  p->dev.maps = static_cast<const unsigned char*>(p->d_maps);
  char* base = static_cast<char*>(p->d_tables);
  size_t cur = 0;
  int rc;
  if ((rc = upload(sc.blocks, base, cur, &p->dev.blocks))) return rc;
  if ((rc = upload(sc.segs, base, cur, &p->dev.segs))) return rc;
  if ((rc = upload(sc.groups, base, cur, &p->dev.groups))) return rc;
  if ((rc = upload(sc.p1, base, cur, &p->dev.p1))) return rc;
  if ((rc = upload(sc.runs, base, cur, &p->dev.runs))) return rc;
  if ((rc = upload(sc.p2, base, cur, &p->dev.p2))) return rc;
  if ((rc = upload(sc.pf, base, cur, &p->dev.pf))) return rc;
  if ((rc = upload(sc.diag, base, cur, &p->dev.diag))) return rc;
  if ((rc = upload(sc.elem, base, cur, &p->dev.elem))) return rc;
  p->dev.n_elem = (int)sc.elem.size();
  p->dev.ws = p->d_ws;
  p->dev.n_blocks = (int)sc.blocks.size();
  p->dev.n_p1 = (int)sc.p1.size();
  p->dev.n_p2 = (int)sc.p2.size();
  p->dev.n_pf = (int)sc.pf.size();
  p->dev.max_block_elems = sc.max_block_elems;
  p->dev.paired = sc.paired ? 1 : 0;
  p->dev.nvec = sc.nvec;
  p->dev.nvec_active = 1;
  p->dev.ld_psi = p->dev.ld_out = sc.psi_len;
  if (sc.psi_len > 0) {
    HPSI_CUDA(cudaMalloc(&p->d_psi_stage, (size_t)sc.psi_len * sizeof(double)));
    HPSI_CUDA(cudaMalloc(&p->d_out_stage, (size_t)sc.psi_len * sizeof(double)));
  }
  return HPSI_OK;
}

void free_plan(hpsi_plan_t* p) {
  if (!p) return;
  if (p->device_ok) {              // whatever upload_schedule / hpsi_davidson / hpsi_truncate got as far as allocating
    cudaFree(p->d_tables);
    cudaFree(p->d_ws);
    cudaFree(p->d_maps);
    cudaFree(p->d_psi_stage);
    cudaFree(p->d_out_stage);
    cudaFree(p->d_dav);
    cudaFree(p->d_svd);
    cudaFreeHost(p->h_dav);
    if (p->dav_side) cudaStreamDestroy(p->dav_side);
    for (auto& e : p->dav_ev) if (e) cudaEventDestroy(e);
    cudaGetLastError();
  }
  delete p;
}

// Tensor maps of every operand matrix (plan.h MapSpec): 2-D FP64 tensor {cols, rows} with row pitch ld, box
// {box_cols, box_rows}, 128-byte swizzle (64-byte for the 8-column boxes of transposed blocks), zero fill outside the matrix.  The encoder is a driver entry point fetched
// through the runtime, so the library does not link libcuda.
typedef CUresult (*tmap_encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                   const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                   CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int encode_maps(hpsi_plan_t* p) {
  static_assert(sizeof(CUtensorMap) == TMAP_BYTES, "CUtensorMap size");
  const std::vector<MapSpec>& specs = p->sc.maps;
  if (specs.empty()) return HPSI_OK;
  tmap_encode_fn enc = nullptr;
  cudaDriverEntryPointQueryResult qr;
  HPSI_CUDA(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", reinterpret_cast<void**>(&enc), cudaEnableDefault, &qr));
  if (!enc || qr != cudaDriverEntryPointSuccess) { set_error("cuTensorMapEncodeTiled not available in this driver"); return HPSI_ECUDA; }
  std::vector<CUtensorMap> host(specs.size());
  for (size_t i = 0; i < specs.size(); ++i) {
    const MapSpec& m = specs[i];
    const double* base = m.base == BASE_A ? p->dev.a : (m.base == BASE_B ? p->dev.b : p->d_ws);
    const cuuint64_t dims[2] = {(cuuint64_t)m.cols, (cuuint64_t)m.rows};
    const cuuint64_t strides[1] = {(cuuint64_t)m.ld * 8};
    const cuuint32_t box[2] = {(cuuint32_t)m.box_cols, (cuuint32_t)m.box_rows};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(&host[i], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double*>(base + m.off), dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, m.box_cols * 8 == 64 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_128B,
                     CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
      char buf[200];
      snprintf(buf, sizeof buf, "cuTensorMapEncodeTiled failed (%d) for a %d x %d matrix with ld %d", (int)r, m.rows, m.cols, m.ld);
      set_error(buf);
      return HPSI_ECUDA;
    }
  }
  HPSI_CUDA(cudaMemcpy(p->d_maps, host.data(), host.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice));
  return HPSI_OK;
}

}  // namespace hpsi

extern "C" int hpsi_bind(hpsi_plan_t* p, const double* a_dev, const double* b_dev) {
  if (!p) { set_error("null plan"); return HPSI_EINVAL; }
  if (p->host_only) { set_error("host-only plan cannot bind device arenas"); return HPSI_ESTATE; }
  bool need_a = false, need_b = false;
  for (const Seg& s : p->sc.segs) { (void)s; need_a = need_b = true; break; }
  if ((need_a && !a_dev) || (need_b && !b_dev)) { set_error("null operator arena"); return HPSI_EINVAL; }
  p->dev.a = a_dev;
  p->dev.b = b_dev;
  p->aligned16 = p->sc.aligned16 && ((reinterpret_cast<uintptr_t>(a_dev) & 15) == 0) &&
                 ((reinterpret_cast<uintptr_t>(b_dev) & 15) == 0);
  if (p->aligned16) {
    int rc = encode_maps(p);
    if (rc != HPSI_OK) return rc;
  }
  p->bound = true;
  return HPSI_OK;
}

extern "C" int hpsi_plan(const hpsi_sectors_t* sectors, const hpsi_terms_t* terms, uint32_t flags,
                         hpsi_plan_t** plan_out) {
  return hpsi_plan_ex(sectors, terms, flags, nullptr, plan_out);
}

extern "C" int hpsi_plan_ex(const hpsi_sectors_t* sectors, const hpsi_terms_t* terms, uint32_t flags,
                            const hpsi_plan_options_t* options, hpsi_plan_t** plan_out) {
  if (!plan_out) { set_error("null plan_out"); return HPSI_EINVAL; }
  *plan_out = nullptr;
  PlanOptions opt;
  if (options) {
    if (options->struct_bytes < sizeof(hpsi_plan_options_t)) { set_error("hpsi_plan_options_t.struct_bytes too small"); return HPSI_EINVAL; }
    opt.shard_of_term = options->shard_of_term;
    opt.shard_index = options->shard_index;
    opt.p1_stages_per_unit = options->p1_stages_per_unit;
    opt.p2_waves = options->p2_waves;
    opt.p2_min_unit_dmma = options->p2_min_unit_dmma;
    opt.n_vectors = options->n_vectors;
  }
  hpsi_plan_t* p = new (std::nothrow) hpsi_plan_t();
  if (!p) { set_error("out of host memory"); return HPSI_ENOMEM; }
  p->host_only = (flags & HPSI_PLAN_HOST_ONLY) != 0;
  int rc = HPSI_OK;
  try {
    if (!p->host_only) {
      int dev = 0;
      cudaError_t e = cudaGetDevice(&dev);
      if (e == cudaSuccess) e = cudaDeviceGetAttribute(&p->n_sm, cudaDevAttrMultiProcessorCount, dev);
      if (e == cudaSuccess) e = kernels_init();
      if (e != cudaSuccess) {
        rc = cuda_fail(e, "device initialisation (no CPU fallback exists)");
        free_plan(p);          // device_ok is still false: nothing to free on the device
        return rc;
      }
      p->device_ok = true;
    }
    std::string err;
    rc = build_schedule(sectors, terms, flags, p->n_sm, opt, &p->sc, &err);
    if (rc != HPSI_OK) { set_error(err); free_plan(p); return rc; }
    p->n_left = sectors->n_left;
    p->n_right = sectors->n_right;
    if (!p->host_only) {
      rc = upload_schedule(p);
      if (rc != HPSI_OK) { free_plan(p); return rc; }
      if (terms->a_data || terms->b_data || p->sc.segs.empty()) {
        rc = hpsi_bind(p, terms->a_data, terms->b_data);
        if (rc != HPSI_OK) { free_plan(p); return rc; }
      }
    }
  } catch (const std::bad_alloc&) {
    set_error("out of host memory while planning");
    free_plan(p);              // frees whatever device buffers were already allocated
    return HPSI_ENOMEM;
  }
  *plan_out = p;
  return HPSI_OK;
}

extern "C" int hpsi_shard_terms(const hpsi_sectors_t* sectors, const hpsi_terms_t* terms, const int32_t* bundle_of_term,
                                int32_t shard_count, int32_t* shard_of_term, int64_t* shard_flops) {
  if (!sectors || !terms || !shard_of_term) { set_error("null argument"); return HPSI_EINVAL; }
  if (shard_count < 1) { set_error("shard_count < 1"); return HPSI_EINVAL; }
  try {
    std::vector<int64_t> flops;
    std::string err;
    int rc = term_useful_flops(sectors, terms, &flops, &err);
    if (rc != HPSI_OK) { set_error(err); return rc; }
    const int T = terms->n_terms;
    // bundles: first term of the bundle is its representative
    struct Bundle { int64_t flops; int32_t first; std::vector<int32_t> terms; };
    std::vector<Bundle> bundles;
    if (bundle_of_term) {
      std::vector<std::pair<int32_t, int32_t>> key(T);
      for (int t = 0; t < T; ++t) key[t] = {bundle_of_term[t], t};
      std::sort(key.begin(), key.end());
      for (int i = 0; i < T; ++i) {
        if (i == 0 || key[i].first != key[i - 1].first) bundles.push_back({0, key[i].second, {}});
        bundles.back().flops += flops[key[i].second];
        bundles.back().terms.push_back(key[i].second);
      }
    } else {
      for (int t = 0; t < T; ++t) bundles.push_back({flops[t], t, {t}});
    }
    std::stable_sort(bundles.begin(), bundles.end(), [](const Bundle& x, const Bundle& y) {
      if (x.flops != y.flops) return x.flops > y.flops;
      return x.first < y.first;
    });
    std::vector<int64_t> load(shard_count, 0);
    for (const Bundle& b : bundles) {
      int best = 0;
      for (int s = 1; s < shard_count; ++s) if (load[s] < load[best]) best = s;
      load[best] += b.flops;
      for (int32_t t : b.terms) shard_of_term[t] = best;
    }
    if (shard_flops) for (int s = 0; s < shard_count; ++s) shard_flops[s] = load[s];
  } catch (const std::bad_alloc&) {
    set_error("out of host memory in hpsi_shard_terms");
    return HPSI_ENOMEM;
  }
  return HPSI_OK;
}

extern "C" int hpsi_layout_blocks(int32_t n_sectors, const int32_t* d, int64_t n_blocks, hpsi_opblock_t* blocks,
                                  const uint8_t* transposed, int64_t* arena_len) {
  if (n_sectors < 0 || n_blocks < 0 || (n_sectors > 0 && !d) || (n_blocks > 0 && !blocks) || !arena_len) {
    set_error("bad argument"); return HPSI_EINVAL;
  }
  int64_t off = 0;
  for (int64_t i = 0; i < n_blocks; ++i) {
    hpsi_opblock_t& e = blocks[i];
    if (e.row < 0 || e.row >= n_sectors || e.col < 0 || e.col >= n_sectors) { set_error("block sector index out of range"); return HPSI_EINVAL; }
    if (e.ld == -1) continue;                             // shares another descriptor's storage
    const bool tr = transposed && transposed[i];
    const int64_t srows = tr ? d[e.col] : d[e.row], scols = tr ? d[e.row] : d[e.col];
    e.ld = sector_up((int)scols);
    e.offset = off;
    off = (off + srows * e.ld + 3) & ~(int64_t)3;
  }
  *arena_len = off;
  return HPSI_OK;
}

extern "C" int hpsi_set_task_coefficients(hpsi_plan_t* p, const double* coef_host, int64_t n, void* cuda_stream) {
  if (!p || !coef_host) { set_error("null argument"); return HPSI_EINVAL; }
  Schedule& sc = p->sc;
  if (n != (int64_t)sc.segs.size()) { set_error("coefficient count != number of tasks (HPSI_Q_N_TASKS)"); return HPSI_EINVAL; }
  for (int64_t i = 0; i < n; ++i) sc.segs[i].coef = coef_host[i];
  for (DiagTask& t : sc.diag) t.coef = coef_host[t.seg];
  if (!p->host_only) {
    // Stream-ordered update of the device tables.  The sources are pageable plan-owned vectors: cudaMemcpyAsync stages
    // them before it returns, and the copies run on `cuda_stream` after whatever was enqueued there before.
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (!sc.segs.empty())
      HPSI_CUDA(cudaMemcpyAsync(const_cast<Seg*>(p->dev.segs), sc.segs.data(), sc.segs.size() * sizeof(Seg), cudaMemcpyHostToDevice, st));
    if (!sc.diag.empty())
      HPSI_CUDA(cudaMemcpyAsync(const_cast<DiagTask*>(p->dev.diag), sc.diag.data(), sc.diag.size() * sizeof(DiagTask), cudaMemcpyHostToDevice, st));
  }
  return HPSI_OK;
}

extern "C" void hpsi_destroy(hpsi_plan_t* p) { free_plan(p); }

extern "C" int hpsi_apply(hpsi_plan_t* p, const double* psi_dev, double* out_dev, void* cuda_stream) {
  return hpsi::apply_impl(p, psi_dev, out_dev, false, cuda_stream);
}

extern "C" int hpsi_apply_multi(hpsi_plan_t* p, const double* psi_dev, int64_t ld_psi, double* out_dev, int64_t ld_out,
                                int32_t n_vectors, void* cuda_stream) {
  if (!p) { set_error("null plan"); return HPSI_EINVAL; }
  if (n_vectors < 1 || n_vectors > p->sc.nvec) { set_error("n_vectors outside 1 .. hpsi_plan_options_t.n_vectors of the plan"); return HPSI_EINVAL; }
  if (ld_psi < p->sc.psi_len || ld_out < p->sc.psi_len) { set_error("vector stride below psi_length"); return HPSI_EINVAL; }
  if (psi_dev && out_dev) {                      // the two sets of vectors must not overlap
    const double *a0 = psi_dev, *a1 = psi_dev + (n_vectors - 1) * ld_psi + p->sc.psi_len;
    const double *b0 = out_dev, *b1 = out_dev + (n_vectors - 1) * ld_out + p->sc.psi_len;
    if (a0 < b1 && b0 < a1 && p->sc.psi_len > 0) { set_error("psi and out must not overlap"); return HPSI_EINVAL; }
  }
  return hpsi::apply_impl(p, psi_dev, out_dev, false, cuda_stream, nullptr, nullptr, n_vectors, ld_psi, ld_out);
}
int hpsi::apply_impl(hpsi_plan_t* p, const double* psi_dev, double* out_dev, bool accumulate, void* cuda_stream,
                     const double* nrm2_dev, double* normalized_dev, int n_vectors, int64_t ld_psi, int64_t ld_out) {
  if (!p) { set_error("null plan"); return HPSI_EINVAL; }
  if (p->host_only) { set_error("host-only plan: hpsi_apply needs a CUDA device (no CPU fallback)"); return HPSI_ESTATE; }
  if (!p->bound) { set_error("operator arenas not bound (hpsi_bind)"); return HPSI_ESTATE; }
  if (p->sc.psi_len == 0) return HPSI_OK;
  if (!psi_dev || !out_dev) { set_error("null psi/out"); return HPSI_EINVAL; }
  if (psi_dev == out_dev) { set_error("psi and out must not alias"); return HPSI_EINVAL; }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  DevSchedule dv = p->dev;                       // per-call view: how many vectors, how far apart
  dv.nvec_active = n_vectors;
  dv.ld_psi = ld_psi > 0 ? ld_psi : p->sc.psi_len;
  dv.ld_out = ld_out > 0 ? ld_out : p->sc.psi_len;
  launch_prep(dv, psi_dev, nrm2_dev, normalized_dev, st);
  launch_p1(dv, p->aligned16, st);
  launch_p2(dv, p->aligned16, st);
  launch_pf(dv, p->aligned16, st);
  launch_reduce(dv, out_dev, accumulate, st);
  HPSI_CUDA(cudaGetLastError());
  return HPSI_OK;
}

extern "C" int hpsi_apply_profiled(hpsi_plan_t* p, const double* psi_dev, double* out_dev, void* cuda_stream,
                                   float* ms_host) {
  if (!p || !ms_host) { set_error("null argument"); return HPSI_EINVAL; }
  if (p->host_only) { set_error("host-only plan: hpsi_apply_profiled needs a CUDA device"); return HPSI_ESTATE; }
  if (!p->bound) { set_error("operator arenas not bound (hpsi_bind)"); return HPSI_ESTATE; }
  if (!psi_dev || !out_dev || psi_dev == out_dev) { set_error("bad psi/out"); return HPSI_EINVAL; }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  EventSet<5> ev;
  HPSI_CUDA(ev.create());
  HPSI_CUDA(cudaEventRecord(ev[0], st));
  launch_prep(p->dev, psi_dev, nullptr, nullptr, st);
  HPSI_CUDA(cudaEventRecord(ev[1], st));
  launch_p1(p->dev, p->aligned16, st);
  HPSI_CUDA(cudaEventRecord(ev[2], st));
  launch_p2(p->dev, p->aligned16, st);
  launch_pf(p->dev, p->aligned16, st);                 // fused units are timed with the second GEMM
  HPSI_CUDA(cudaEventRecord(ev[3], st));
  launch_reduce(p->dev, out_dev, false, st);
  HPSI_CUDA(cudaEventRecord(ev[4], st));
  HPSI_CUDA(cudaEventSynchronize(ev[4]));
  for (int i = 0; i < 4; ++i) HPSI_CUDA(cudaEventElapsedTime(&ms_host[i], ev[i], ev[i + 1]));
  HPSI_CUDA(cudaGetLastError());
  return HPSI_OK;
}

extern "C" int hpsi_apply_host(hpsi_plan_t* p, const double* psi_host, double* out_host, void* cuda_stream) {
  if (!p) { set_error("null plan"); return HPSI_EINVAL; }
  if (p->host_only) { set_error("host-only plan: hpsi_apply_host needs a CUDA device (no CPU fallback)"); return HPSI_ESTATE; }
  if (p->sc.psi_len == 0) return HPSI_OK;
  if (!psi_host || !out_host) { set_error("null psi/out"); return HPSI_EINVAL; }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const size_t bytes = (size_t)p->sc.psi_len * sizeof(double);
  HPSI_CUDA(cudaMemcpyAsync(p->d_psi_stage, psi_host, bytes, cudaMemcpyHostToDevice, st));
  int rc = hpsi_apply(p, p->d_psi_stage, p->d_out_stage, cuda_stream);
  if (rc != HPSI_OK) return rc;
  HPSI_CUDA(cudaMemcpyAsync(out_host, p->d_out_stage, bytes, cudaMemcpyDeviceToHost, st));
  HPSI_CUDA(cudaStreamSynchronize(st));
  return HPSI_OK;
}

extern "C" int hpsi_sum_shards(const double* parts_dev, int32_t n_parts, int64_t n, double* out_dev, void* cuda_stream) {
  if (n_parts < 1 || n < 0) { set_error("bad shard count / length"); return HPSI_EINVAL; }
  if (n == 0) return HPSI_OK;
  if (!parts_dev || !out_dev) { set_error("null argument"); return HPSI_EINVAL; }
  if (out_dev > parts_dev - n && out_dev < parts_dev + (int64_t)n_parts * n && out_dev != parts_dev) {
    set_error("out overlaps parts (only out == parts, i.e. in place over shard 0, is allowed)"); return HPSI_EINVAL;
  }
  launch_sum_shards(parts_dev, n_parts, n, out_dev, static_cast<cudaStream_t>(cuda_stream));
  HPSI_CUDA(cudaGetLastError());
  return HPSI_OK;
}

extern "C" int hpsi_diagonal(hpsi_plan_t* p, double* diag_dev, void* cuda_stream) {
  if (!p) { set_error("null plan"); return HPSI_EINVAL; }
  if (p->host_only) { set_error("host-only plan: hpsi_diagonal needs a CUDA device"); return HPSI_ESTATE; }
  if (!p->bound) { set_error("operator arenas not bound (hpsi_bind)"); return HPSI_ESTATE; }
  if (p->sc.psi_len == 0) return HPSI_OK;
  if (!diag_dev) { set_error("null diag"); return HPSI_EINVAL; }
  launch_diag(p->dev, diag_dev, static_cast<cudaStream_t>(cuda_stream));
  HPSI_CUDA(cudaGetLastError());
  return HPSI_OK;
}

extern "C" int hpsi_query(const hpsi_plan_t* p, int what, void* out, size_t bytes) {
  if (!p || !out) { set_error("null argument"); return HPSI_EINVAL; }
  const Schedule& sc = p->sc;
  auto put_i64 = [&](int64_t v) -> int {
    if (bytes < sizeof(int64_t)) { set_error("hpsi_query: buffer too small"); return HPSI_EINVAL; }
    memcpy(out, &v, sizeof v);
    return HPSI_OK;
  };
  switch (what) {
    case HPSI_Q_PSI_LENGTH: return put_i64(sc.psi_len);
    case HPSI_Q_N_PSI_BLOCKS: return put_i64((int64_t)sc.blocks.size());
    case HPSI_Q_PSI_BLOCKS: {
      if (bytes < sc.blocks.size() * sizeof(hpsi_psi_block_t)) { set_error("hpsi_query: buffer too small"); return HPSI_EINVAL; }
      hpsi_psi_block_t* o = static_cast<hpsi_psi_block_t*>(out);
      for (size_t i = 0; i < sc.blocks.size(); ++i)
        o[i] = {sc.blocks[i].left, sc.blocks[i].right, sc.blocks[i].rows, sc.blocks[i].cols, sc.blocks[i].off};
      return HPSI_OK;
    }
    case HPSI_Q_N_TASKS: return put_i64((int64_t)sc.segs.size());
    case HPSI_Q_USEFUL_FLOPS: return put_i64(sc.useful_flops);
    case HPSI_Q_USEFUL_FLOPS_P1: return put_i64(sc.useful_flops_p1);
    case HPSI_Q_ISSUED_FLOPS: return put_i64(sc.issued_flops);
    case HPSI_Q_ISSUED_FLOPS_P1: return put_i64(sc.issued_flops_p1);
    case HPSI_Q_CRITICAL_FLOPS: return put_i64(sc.critical_flops);
    case HPSI_Q_OPERATOR_BYTES: return put_i64(sc.operator_bytes);
    case HPSI_Q_WORKSPACE_BYTES: return put_i64(sc.ws_len * 8);
    case HPSI_Q_N_GROUPS: return put_i64((int64_t)sc.groups.size());
    case HPSI_Q_N_P1_UNITS: return put_i64((int64_t)sc.p1.size());
    case HPSI_Q_N_P2_UNITS: return put_i64((int64_t)sc.p2.size());
    case HPSI_Q_N_ORDER1_TASKS: return put_i64(sc.n_order1);
    case HPSI_Q_LAUNCHES_PER_APPLY:
      return put_i64((sc.blocks.empty() ? 0 : 2) + (sc.p1.empty() ? 0 : 1) + (sc.p2.empty() ? 0 : 1) + (sc.pf.empty() ? 0 : 1));
    case HPSI_Q_N_FUSED_UNITS: return put_i64((int64_t)sc.pf.size());
    case HPSI_Q_N_FUSED_TASKS: { int64_t n = 0; for (const Group& g : sc.groups) if (g.fused) n += g.tcount; return put_i64(n); }
    case HPSI_Q_ALIGNED16: return put_i64(p->host_only ? sc.aligned16 : p->aligned16);
    case HPSI_Q_INTERMEDIATE_BYTES: return put_i64(sc.intermediate_bytes);
    case HPSI_Q_PSI_ROWS: { int64_t n = 0; for (const PsiBlk& b : sc.blocks) n += b.rows; return put_i64(n); }
    case HPSI_Q_ISO_CAPACITY: { int64_t n = 0; for (const PsiBlk& b : sc.blocks) n += (int64_t)std::min(b.rows, b.cols) * b.rows; return put_i64(n); }
    case HPSI_Q_PSI_COLS: { int64_t n = 0; for (const PsiBlk& b : sc.blocks) n += b.cols; return put_i64(n); }
    case HPSI_Q_ISO_CAPACITY_RIGHT: { int64_t n = 0; for (const PsiBlk& b : sc.blocks) n += (int64_t)std::min(b.rows, b.cols) * b.cols; return put_i64(n); }
    case HPSI_Q_SVD_SWEEPS: return put_i64(p->svd_sweeps);
    case HPSI_Q_SVD_LAUNCHES: return put_i64(p->svd_launches);
    case HPSI_Q_N_TERMS_PLANNED: return put_i64(sc.n_terms_planned);
    case HPSI_Q_N_VECTORS: return put_i64(sc.nvec);
    case HPSI_Q_TUNING: {
      if (bytes < sizeof sc.tuning) { set_error("hpsi_query: buffer too small"); return HPSI_EINVAL; }
      memcpy(out, sc.tuning, sizeof sc.tuning);
      return HPSI_OK;
    }
    case HPSI_Q_PREFERRED_LAYOUT: {
      if (bytes < sizeof(hpsi_layout_t)) { set_error("hpsi_query: buffer too small"); return HPSI_EINVAL; }
      const hpsi_layout_t lay = {4, 4, 2, 2, 16, 8};
      memcpy(out, &lay, sizeof lay);
      return HPSI_OK;
    }
    case HPSI_Q_TASKS: {
      if (bytes < sc.tasks.size() * sizeof(hpsi_task_t)) { set_error("hpsi_query: buffer too small"); return HPSI_EINVAL; }
      if (!sc.tasks.empty()) memcpy(out, sc.tasks.data(), sc.tasks.size() * sizeof(hpsi_task_t));
      return HPSI_OK;
    }
    default: set_error("hpsi_query: unknown item"); return HPSI_EINVAL;
  }
}

extern "C" int hpsi_debug_interpret(const hpsi_plan_t* p, const double* a_host, const double* b_host,
                                    const double* psi_host, double* out_host) {
  return hpsi_debug_interpret_multi(p, a_host, b_host, psi_host, out_host, 1);
}

extern "C" int hpsi_debug_interpret_multi(const hpsi_plan_t* p, const double* a_host, const double* b_host,
                                          const double* psi_host, double* out_host, int32_t n_vectors) {
  if (!p) { set_error("null plan"); return HPSI_EINVAL; }
  if (n_vectors < 1 || n_vectors > p->sc.nvec) { set_error("n_vectors outside 1 .. the plan's n_vectors"); return HPSI_EINVAL; }
  if (p->sc.psi_len > 0 && (!psi_host || !out_host)) { set_error("null psi/out"); return HPSI_EINVAL; }
  if (!p->sc.segs.empty() && (!a_host || !b_host)) { set_error("null arena"); return HPSI_EINVAL; }
  try {
    interpret_schedule(p->sc, a_host, b_host, psi_host, out_host, n_vectors);
  } catch (const std::bad_alloc&) {
    set_error("out of host memory in interpreter");
    return HPSI_ENOMEM;
  }
  return HPSI_OK;
}
