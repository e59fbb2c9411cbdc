// boa_stream.cu — the streaming front end of include/boa.h (PAPER Fig. 2).
//
// "Buffer chunks in parallel, compress in parallel, pre-load the next compressor set": the input is cut into groups of
// `group_chunks` chunks; every group becomes one complete BOA1 container (a shard) and the shards are concatenated.
// While the step kernels work on group k (boa_compress / boa_decompress on device buffers, on the caller's stream),
// a second CUDA stream brings group k+1 from pinned host memory into the other device buffer and takes shard k-1
// back, so the host <-> device traffic of a group hides behind the computation of its neighbours.
// Built only on the public entry points of boa_api.cu and the container helpers; no kernel of its own.
#include "../../include/boa.h"

#include <cuda_runtime.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "container.h"

using namespace boa;

namespace {

// two device buffers + two pinned host buffers per direction, one copy stream, events
struct Lanes {
  uint8_t *d_in[2] = {nullptr, nullptr}, *d_out[2] = {nullptr, nullptr};
  uint8_t *h_in[2] = {nullptr, nullptr}, *h_out[2] = {nullptr, nullptr};
  cudaStream_t cp = nullptr;
  cudaEvent_t in_ready[2] = {nullptr, nullptr}, out_ready[2] = {nullptr, nullptr};
  bool ok = true;

  Lanes(size_t in_bytes, size_t out_bytes) {
    auto chk = [&](cudaError_t e) { if (e != cudaSuccess) { (void)cudaGetLastError(); ok = false; } };
    chk(cudaStreamCreateWithFlags(&cp, cudaStreamNonBlocking));
    for (int i = 0; i < 2 && ok; ++i) {
      chk(cudaMalloc(&d_in[i], std::max<size_t>(in_bytes, 1)));
      chk(cudaMalloc(&d_out[i], std::max<size_t>(out_bytes, 1)));
      chk(cudaHostAlloc(&h_in[i], std::max<size_t>(in_bytes, 1), cudaHostAllocDefault));
      chk(cudaHostAlloc(&h_out[i], std::max<size_t>(out_bytes, 1), cudaHostAllocDefault));
      chk(cudaEventCreateWithFlags(&in_ready[i], cudaEventDisableTiming));
      chk(cudaEventCreateWithFlags(&out_ready[i], cudaEventDisableTiming));
    }
  }
  ~Lanes() {
    if (cp) cudaStreamSynchronize(cp);
    for (int i = 0; i < 2; ++i) {
      if (d_in[i]) cudaFree(d_in[i]);
      if (d_out[i]) cudaFree(d_out[i]);
      if (h_in[i]) cudaFreeHost(h_in[i]);
      if (h_out[i]) cudaFreeHost(h_out[i]);
      if (in_ready[i]) cudaEventDestroy(in_ready[i]);
      if (out_ready[i]) cudaEventDestroy(out_ready[i]);
    }
    if (cp) cudaStreamDestroy(cp);
    (void)cudaGetLastError();
  }
};

bool on_device(const void* p) {
  if (!p) return false;
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { (void)cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeDevice;
}

#define STREAM_CUDA_TRY(expr)                                              \
  do {                                                                     \
    if ((expr) != cudaSuccess) { (void)cudaGetLastError(); return BOA_E_CUDA; } \
  } while (0)

// length of the BOA1 container that starts at p (host), from its header and size index; 0 if it does not fit in `avail`
size_t shard_length(const uint8_t* p, size_t avail, uint64_t* n_out) {
  if (avail < kHeaderBytes + 4) return 0;
  Header h;
  if (!parse_header(p, h)) return 0;
  const size_t ib = index_bytes(h.n_chunks);
  if (avail < ib) return 0;
  const uint8_t* sp = p + kHeaderBytes + first_padded(h.n_chunks);
  uint64_t total = ib;
  for (uint64_t i = 0; i < h.n_chunks; ++i) total += get_u32(sp + 4 * i);
  if (total > avail) return 0;
  if (n_out) *n_out = h.n;
  return (size_t)total;
}

}  // namespace

extern "C" size_t boa_stream_bound(size_t n, size_t chunk_bytes, size_t group_chunks) {
  if (chunk_bytes == 0 || group_chunks == 0) return 0;
  const size_t group_bytes = chunk_bytes * group_chunks;
  const size_t full = n / group_bytes, rest = n - full * group_bytes;
  return full * boa_compress_bound(group_bytes, chunk_bytes) + (rest ? boa_compress_bound(rest, chunk_bytes) : 0);
}

extern "C" int boa_stream_compress(boa_model* m, const uint8_t* in, size_t n, size_t chunk_bytes, size_t group_chunks,
                                   uint8_t* out, size_t* out_len, uint64_t* shard_len, size_t* n_shards, void* cuda_stream) {
  if (!m || !out_len || chunk_bytes == 0 || chunk_bytes > boa::kMaxChunkBytes || group_chunks == 0 || (n && (!in || !out)))
    return BOA_E_ARG;
  if (on_device(in) || on_device(out)) return BOA_E_ARG;     // the streaming entry points take host buffers
  const size_t group_bytes = chunk_bytes * group_chunks;
  const size_t groups = n ? (n + group_bytes - 1) / group_bytes : 0;
  const size_t shard_cap = n_shards ? *n_shards : 0;
  if (shard_len && shard_cap < groups) return BOA_E_CAPACITY;
  const size_t capacity = *out_len;
  *out_len = 0;
  if (n_shards) *n_shards = 0;
  if (groups == 0) return BOA_OK;

  const size_t in_cap = std::min(group_bytes, n), out_cap = boa_compress_bound(in_cap, chunk_bytes);
  Lanes L(in_cap, out_cap);
  if (!L.ok) return BOA_E_NOMEM;
  cudaStream_t user = static_cast<cudaStream_t>(cuda_stream);
  auto group_len = [&](size_t k) { return std::min(group_bytes, n - k * group_bytes); };
  auto preload = [&](size_t k) -> int {     // Fig. 2, red: group k -> pinned lane -> device lane, on the copy stream
    const int b = (int)(k & 1);
    memcpy(L.h_in[b], in + k * group_bytes, group_len(k));
    STREAM_CUDA_TRY(cudaMemcpyAsync(L.d_in[b], L.h_in[b], group_len(k), cudaMemcpyHostToDevice, L.cp));
    STREAM_CUDA_TRY(cudaEventRecord(L.in_ready[b], L.cp));
    return BOA_OK;
  };
  size_t written = 0;
  size_t pending_len[2] = {0, 0};            // shard on its way back through pinned lane b
  auto collect = [&](size_t k) -> int {      // shard k: pinned lane -> the caller's buffer
    const int b = (int)(k & 1);
    STREAM_CUDA_TRY(cudaEventSynchronize(L.out_ready[b]));
    if (written + pending_len[b] > capacity) return BOA_E_CAPACITY;
    memcpy(out + written, L.h_out[b], pending_len[b]);
    if (shard_len) shard_len[k] = pending_len[b];
    written += pending_len[b];
    return BOA_OK;
  };

  int rc = preload(0);
  for (size_t k = 0; k < groups && rc == BOA_OK; ++k) {
    const int b = (int)(k & 1);
    if (k + 1 < groups) rc = preload(k + 1);                 // flies while group k is compressed
    if (rc != BOA_OK) break;
    STREAM_CUDA_TRY(cudaStreamWaitEvent(user, L.in_ready[b], 0));
    size_t len = out_cap;
    rc = boa_compress(m, L.d_in[b], group_len(k), chunk_bytes, L.d_out[b], &len, cuda_stream);   // Fig. 2, green
    if (rc != BOA_OK) break;
    // boa_compress returns with its work complete: the shard can leave on the copy stream while group k+1 runs
    pending_len[b] = len;
    STREAM_CUDA_TRY(cudaMemcpyAsync(L.h_out[b], L.d_out[b], len, cudaMemcpyDeviceToHost, L.cp));
    STREAM_CUDA_TRY(cudaEventRecord(L.out_ready[b], L.cp));
    if (k >= 1) rc = collect(k - 1);
  }
  if (rc == BOA_OK) rc = collect(groups - 1);
  if (rc != BOA_OK) return rc;
  *out_len = written;
  if (n_shards) *n_shards = groups;
  return BOA_OK;
}

extern "C" int boa_stream_decompressed_size(const uint8_t* in, size_t in_len, size_t* n, size_t* n_shards) {
  if ((!in && in_len) || !n) return BOA_E_ARG;
  size_t off = 0, total = 0, shards = 0;
  while (off < in_len) {
    uint64_t ni = 0;
    const size_t len = shard_length(in + off, in_len - off, &ni);
    if (len == 0) return BOA_E_FORMAT;
    off += len; total += (size_t)ni; ++shards;
  }
  *n = total;
  if (n_shards) *n_shards = shards;
  return BOA_OK;
}

extern "C" int boa_stream_decompress(boa_model* m, const uint8_t* in, size_t in_len, uint8_t* out, size_t* out_len,
                                     void* cuda_stream) {
  if (!m || !out_len || (in_len && !in) || on_device(in) || on_device(out)) return BOA_E_ARG;
  // walk the shards once on the host: offsets, lengths, decoded sizes
  struct Shard { size_t off, len, n, out_off; };
  std::vector<Shard> sh;
  size_t off = 0, total = 0, max_len = 0, max_n = 0;
  while (off < in_len) {
    uint64_t ni = 0;
    const size_t len = shard_length(in + off, in_len - off, &ni);
    if (len == 0) return BOA_E_FORMAT;
    sh.push_back({off, len, (size_t)ni, total});
    off += len; total += (size_t)ni;
    max_len = std::max(max_len, len); max_n = std::max(max_n, (size_t)ni);
  }
  if (*out_len < total) return BOA_E_CAPACITY;
  if (total && !out) return BOA_E_ARG;
  *out_len = 0;
  if (sh.empty()) return BOA_OK;

  Lanes L(max_len, max_n);
  if (!L.ok) return BOA_E_NOMEM;
  cudaStream_t user = static_cast<cudaStream_t>(cuda_stream);
  auto preload = [&](size_t k) -> int {
    const int b = (int)(k & 1);
    memcpy(L.h_in[b], in + sh[k].off, sh[k].len);
    STREAM_CUDA_TRY(cudaMemcpyAsync(L.d_in[b], L.h_in[b], sh[k].len, cudaMemcpyHostToDevice, L.cp));
    STREAM_CUDA_TRY(cudaEventRecord(L.in_ready[b], L.cp));
    return BOA_OK;
  };
  auto collect = [&](size_t k) -> int {
    const int b = (int)(k & 1);
    STREAM_CUDA_TRY(cudaEventSynchronize(L.out_ready[b]));
    memcpy(out + sh[k].out_off, L.h_out[b], sh[k].n);
    return BOA_OK;
  };
  int rc = preload(0);
  for (size_t k = 0; k < sh.size() && rc == BOA_OK; ++k) {
    const int b = (int)(k & 1);
    if (k + 1 < sh.size()) rc = preload(k + 1);
    if (rc != BOA_OK) break;
    STREAM_CUDA_TRY(cudaStreamWaitEvent(user, L.in_ready[b], 0));
    size_t len = std::max<size_t>(max_n, 1);
    rc = boa_decompress(m, L.d_in[b], sh[k].len, L.d_out[b], &len, cuda_stream);
    if (rc != BOA_OK) break;
    if (len != sh[k].n) { rc = BOA_E_FORMAT; break; }
    STREAM_CUDA_TRY(cudaMemcpyAsync(L.h_out[b], L.d_out[b], std::max<size_t>(len, 1), cudaMemcpyDeviceToHost, L.cp));
    STREAM_CUDA_TRY(cudaEventRecord(L.out_ready[b], L.cp));
    if (k >= 1) rc = collect(k - 1);
  }
  if (rc == BOA_OK) rc = collect(sh.size() - 1);
  if (rc != BOA_OK) return rc;
  *out_len = total;
  return BOA_OK;
}
