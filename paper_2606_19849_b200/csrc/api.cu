// Library-level entry points: version, errors, device info, KV-pool validation and TMA maps.
#include "common.cuh"

#include <cmath>
#include <cstring>

namespace vcs {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}

unsigned long long turn_fraction_q64(double inv_freq) {
  const long double turns = (long double)inv_freq / 6.283185307179586476925286766559L;
  const long double fr = turns - floorl(turns);
  return (unsigned long long)(fr * 18446744073709551616.0L);
}

int device_sm_count() {
  static std::atomic<int> cache[kMaxDevices];
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return 0; }
  const bool cached = dev >= 0 && dev < kMaxDevices;
  int n = cached ? cache[dev].load(std::memory_order_relaxed) : 0;
  if (n > 0) return n;
  if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) { cudaGetLastError(); return 0; }
  if (cached) cache[dev].store(n, std::memory_order_relaxed);
  return n;
}

int validate_pool(const vcs_kv_pool* p, bool need_opaque) {
  if (!p) VCS_FAIL(VCS_EINVAL, "pool is NULL");
  if (!p->k_pages || !p->v_pages || !p->page_len || !p->k_sum) VCS_FAIL(VCS_EINVAL, "pool has a NULL buffer");
  if (p->n_pages <= 0 || p->page_cap <= 0 || p->Hkv <= 0 || p->Hq <= 0 || p->d <= 0)
    VCS_FAIL(VCS_EINVAL, "pool sizes must be positive");
  if (p->Hq % p->Hkv != 0) VCS_FAIL(VCS_EINVAL, "Hq (%d) must be a multiple of Hkv (%d)", p->Hq, p->Hkv);
  if (p->dtype != VCS_F32 && p->dtype != VCS_BF16) VCS_FAIL(VCS_EUNSUPPORTED, "pool dtype %d", p->dtype);
  if (p->d != 64 && p->d != 128) VCS_FAIL(VCS_EUNSUPPORTED, "head_dim %d not in {64,128}", p->d);
  if (p->rope_sections[0] < 0 || p->rope_sections[1] < 0 || p->rope_sections[2] < 0 ||
      p->rope_sections[0] + p->rope_sections[1] + p->rope_sections[2] != p->d / 2)
    VCS_FAIL(VCS_EINVAL, "rope_sections must be non-negative and sum to d/2");
  if (!(p->rope_theta > 0.f)) VCS_FAIL(VCS_EINVAL, "rope_theta must be positive");
  if (!aligned16(p->k_pages) || !aligned16(p->v_pages) || !aligned16(p->k_sum))
    VCS_FAIL(VCS_EALIGN, "pool buffers must be 16-byte aligned");
  if (need_opaque) {
    if (!p->opaque_h) VCS_FAIL(VCS_EINVAL, "pool.opaque_h is NULL (call vcs_pool_init)");
    if (reinterpret_cast<const PoolOpaque*>(p->opaque_h)->magic != kPoolMagic)
      VCS_FAIL(VCS_EINVAL, "pool.opaque_h not initialised (call vcs_pool_init)");
  }
  return VCS_OK;
}

RopeParams rope_params(const vcs_kv_pool* p) {
  RopeParams r;
  const PoolOpaque* o = reinterpret_cast<const PoolOpaque*>(p->opaque_h);
  r.half = p->d / 2;
  for (int m = 0; m < 64; ++m) {
    r.inv_freq[m] = m < r.half ? o->inv_freq[m] : 0.0;
    r.turn_frac[m] = turn_fraction_q64(r.inv_freq[m]);
    r.axis_of[m] = m < r.half ? o->axis_of[m] : 0;
  }
  return r;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (fn) return fn;
  void* sym = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) != cudaSuccess ||
      qres != cudaDriverEntryPointSuccess)
    return nullptr;
  fn = reinterpret_cast<EncodeTiledFn>(sym);
  return fn;
}

// 4-D map over a pool buffer [n_pages][Hkv][page_cap][d] bf16: dims (d, token, head, page),
// box (64 elements = 128 B, 64 tokens, 1, 1), 128-byte swizzle.
static int encode_pool_map(CUtensorMap* map, void* base, const vcs_kv_pool* p) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) VCS_FAIL(VCS_ECUDA, "cuTensorMapEncodeTiled not available from the driver");
  cuuint64_t dims[4] = {(cuuint64_t)p->d, (cuuint64_t)p->page_cap, (cuuint64_t)p->Hkv, (cuuint64_t)p->n_pages};
  cuuint64_t strides[3] = {(cuuint64_t)p->d * 2, (cuuint64_t)p->page_cap * p->d * 2,
                           (cuuint64_t)p->Hkv * p->page_cap * p->d * 2};
  cuuint32_t box[4] = {64, 64, 1, 1};   // 64 d-elements (128 B) x 64 tokens (kAttnKvTile)
  cuuint32_t estr[4] = {1, 1, 1, 1};
  CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, base, dims, strides, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) VCS_FAIL(VCS_ECUDA, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
  return VCS_OK;
}

}  // namespace vcs

using namespace vcs;

extern "C" {

int vcs_version(void) { return VCS_VERSION; }

size_t vcs_sizeof_chunk_call(void) { return sizeof(vcs_chunk_call); }
size_t vcs_sizeof_multi_call(void) { return sizeof(vcs_multi_call); }

const char* vcs_last_error(void) { return g_err; }

int vcs_device_info(int* sm_count_h, int* cc_major_h, int* cc_minor_h, char* name_h, size_t name_bytes) {
  int dev = 0;
  VCS_CUDA_OK(cudaGetDevice(&dev));
  cudaDeviceProp prop;
  VCS_CUDA_OK(cudaGetDeviceProperties(&prop, dev));
  if (sm_count_h) *sm_count_h = prop.multiProcessorCount;
  if (cc_major_h) *cc_major_h = prop.major;
  if (cc_minor_h) *cc_minor_h = prop.minor;
  if (name_h && name_bytes) {
    strncpy(name_h, prop.name, name_bytes - 1);
    name_h[name_bytes - 1] = 0;
  }
  return VCS_OK;
}

// Step a6, vision side (V_vis(t) = { j : t - acn <= j <= t }; readings D11, D12, D14): the
// fully visible pages of chunk t are the sink page, then the pages of chunks max(0, t - W) .. t - 1 in stream
// order; the chunk's own page is the causal self page of the attention call and is not listed.  Host only.
int vcs_visible_set(int32_t t, int32_t W, int32_t sink_page, const int32_t* chunk_pages_h, int32_t n_chunks,
                    int32_t* table_out_h, int32_t table_cap) {
  if (t < 0 || n_chunks < 0 || t > n_chunks || table_cap < 0 || (!chunk_pages_h && n_chunks > 0) || (!table_out_h && table_cap > 0))
    VCS_FAIL(VCS_EINVAL, "visible_set: bad arguments");
  const int32_t lo = W < 0 ? 0 : (t - W > 0 ? t - W : 0);
  const int32_t n = (sink_page >= 0 ? 1 : 0) + (t - lo);
  if (n > table_cap) VCS_FAIL(VCS_ECAP, "visible_set: %d entries do not fit a table of %d", n, table_cap);
  int32_t k = 0;
  if (sink_page >= 0) table_out_h[k++] = sink_page;
  for (int32_t j = lo; j < t; ++j) table_out_h[k++] = chunk_pages_h[j];
  for (int32_t j = k; j < table_cap; ++j) table_out_h[j] = -1;
  return n;
}

// Step a6, query side (readings D14, D21): a query token sees the sink page, the `recent` most
// recent chunk pages and the k retrieved ones.  The table is laid out as [sink][recent ...][k slots], the k slots
// set to -1 for vcs_retrieval_score to fill on the device (topk_pages = table + return value); -1 entries that
// remain (fewer than k eligible chunks) are skipped by the attention kernels.  Host only.
int vcs_visible_set_query(int32_t sink_page, const int32_t* recent_pages_h, int32_t n_recent, int32_t k,
                          int32_t* table_out_h, int32_t table_cap) {
  if (n_recent < 0 || k < 0 || table_cap < 0 || (!recent_pages_h && n_recent > 0) || (!table_out_h && table_cap > 0))
    VCS_FAIL(VCS_EINVAL, "visible_set_query: bad arguments");
  const int64_t n_fixed = (sink_page >= 0 ? 1 : 0) + (int64_t)n_recent;
  if (n_fixed + k > table_cap) VCS_FAIL(VCS_ECAP, "visible_set_query: %lld entries do not fit a table of %d", (long long)(n_fixed + k), table_cap);
  int32_t j = 0;
  if (sink_page >= 0) table_out_h[j++] = sink_page;
  for (int32_t r = 0; r < n_recent; ++r) {
    if (recent_pages_h[r] < 0) VCS_FAIL(VCS_EINVAL, "visible_set_query: negative recent page id");
    table_out_h[j++] = recent_pages_h[r];
  }
  for (; j < table_cap; ++j) table_out_h[j] = -1;
  return (int)n_fixed;
}

// Positions (reading D18; the oracle's O2).  A chunk whose position base is b occupies (b + g t_stride,
// b + r, b + c); the next chunk's base is b + max(G t_stride, Hg, Wg), so that no axis runs backwards.  Text and
// sink tokens sit on the diagonal: token i of a run starting at `start` has (start + i) on all three axes.  Host only.
int vcs_next_position_base(int32_t G, int32_t Hg, int32_t Wg, int32_t t_stride, int32_t base, int32_t* next_base_h) {
  if (G <= 0 || Hg <= 0 || Wg <= 0 || t_stride <= 0 || base < 0 || !next_base_h) VCS_FAIL(VCS_EINVAL, "next_position_base: bad arguments");
  int64_t step = (int64_t)G * t_stride;
  if (Hg > step) step = Hg;
  if (Wg > step) step = Wg;
  if (base + step > 0x7fffffffLL) VCS_FAIL(VCS_ECAP, "next_position_base: position overflows int32");
  *next_base_h = (int32_t)(base + step);
  return VCS_OK;
}

int vcs_text_positions(int32_t start, int32_t n, int32_t* pos3_out_h) {
  if (start < 0 || n < 0 || (!pos3_out_h && n > 0)) VCS_FAIL(VCS_EINVAL, "text_positions: bad arguments");
  if ((int64_t)start + n > 0x7fffffffLL) VCS_FAIL(VCS_ECAP, "text_positions: position overflows int32");
  for (int32_t i = 0; i < n; ++i) pos3_out_h[3 * i] = pos3_out_h[3 * i + 1] = pos3_out_h[3 * i + 2] = start + i;
  return VCS_OK;
}

size_t vcs_pool_opaque_bytes(void) { return sizeof(PoolOpaque) + 64; }

int vcs_pool_init(vcs_kv_pool* p) {
  int rc = validate_pool(p, false);
  if (rc != VCS_OK) return rc;
  if (!p->opaque_h) VCS_FAIL(VCS_EINVAL, "pool.opaque_h is NULL");
  if (reinterpret_cast<uintptr_t>(p->opaque_h) & 63u) VCS_FAIL(VCS_EALIGN, "pool.opaque_h must be 64-byte aligned");
  PoolOpaque* o = reinterpret_cast<PoolOpaque*>(p->opaque_h);
  memset(o, 0, sizeof(*o));
  const int half = p->d / 2;
  int m = 0;
  for (int ax = 0; ax < 3; ++ax)
    for (int i = 0; i < p->rope_sections[ax]; ++i, ++m) o->axis_of[m] = (int8_t)ax;
  for (m = 0; m < half; ++m) o->inv_freq[m] = pow((double)p->rope_theta, -2.0 * m / p->d);
  o->has_tma = 0;
  if (p->dtype == VCS_BF16 && p->d == 128) {
    // TMA maps need a device/driver; without one the pool is still usable by the SIMT kernels.
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) == cudaSuccess && ndev > 0) {
      rc = encode_pool_map(&o->tmap_k, p->k_pages, p);
      if (rc != VCS_OK) return rc;
      rc = encode_pool_map(&o->tmap_v, p->v_pages, p);
      if (rc != VCS_OK) return rc;
      o->has_tma = 1;
    } else {
      cudaGetLastError();
    }
  }
  o->magic = kPoolMagic;
  return VCS_OK;
}

}  // extern "C"
