/* boa.h — C ABI of the B200-native chunk-parallel neural range coder
 * (the hot path of BOA Constrictor, arXiv 2511.11337).
 *
 * Citations: `P:n` = line n of the paper text.  Readings of passages where the paper is
 * silent or garbled are numbered in DESIGN.md ("Readings") and referred to as R#k.
 *
 * The library owns every step of the path: split into chunks, byte embedding + Mamba-1
 * blocks + tied head (Alg. 1; eq. 16-22), softmax (eq. 6), the
 * integer table (eq. 7), the range coder (eq. 8-13) and the .boa container
 * (P:167).  All of it runs in CUDA kernels for sm_100a; there is no CPU fallback — every entry
 * point that needs the GPU returns BOA_E_CUDA when no device is usable.
 *
 * Conventions
 *   - Return value: 0 (BOA_OK) or a negative BOA_E_* code; boa_strerror() names it.  Nothing
 *     throws, aborts or prints.
 *   - "host|device pointer": the library asks the CUDA runtime what the pointer is
 *     (cudaPointerGetAttributes).  Device (or managed) memory is used in place; host memory
 *     (pageable or pinned) is staged through a library-owned device buffer with the copies issued
 *     on `cuda_stream` inside the call (this is what the end-to-end benchmark times).
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  The
 *     library orders its work after everything already enqueued on that stream (it records an event
 *     there and runs on a stream of its own, because the step loop is replayed from CUDA graphs and
 *     the legacy stream cannot be captured) and returns only after all of its work has completed.
 *   - One in-flight call per boa_model handle; different handles may be used concurrently.
 *   - The caller owns all `in`/`out` buffers.  The handle owns the device copy of the weights and
 *     a workspace (stream state, activations, per-stream output scratch) that grows to the largest
 *     job seen and is released by boa_model_free().
 */
#ifndef BOA_H_
#define BOA_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BOA_OK 0
#define BOA_E_ARG (-1)            /* NULL / zero / out-of-range argument                              */
#define BOA_E_FORMAT (-2)         /* bad magic, version, freq_bits or inconsistent lengths            */
#define BOA_E_CRC (-3)            /* index CRC-32 mismatch                                            */
#define BOA_E_MODEL_MISMATCH (-4) /* container fingerprint != this model + this arithmetic            */
#define BOA_E_CAPACITY (-5)       /* output buffer too small                                          */
#define BOA_E_CORRUPT (-6)        /* a stream's payload ended before its symbols were decoded         */
#define BOA_E_CUDA (-7)           /* CUDA runtime error or no usable sm_100 device                    */
#define BOA_E_NOMEM (-8)          /* host or device allocation failed                                 */
#define BOA_E_UNSUPPORTED (-9)    /* model shape outside what the kernels are built for               */

typedef struct boa_model boa_model; /* opaque: device weights + workspace */

/* ---- model ------------------------------------------------------------------------------------
 * boa_model_load: parse a BOAW v1 blob (HOST pointer; layout in DESIGN.md "BOAW") — byte embedding
 * [256][D] (also the tied head), per layer norm_w, W_in, conv_w, conv_b, W_x, W_dt,
 * b_dt, A_log, D_skip, W_out (eq. 20-22) — copy it to the current CUDA device and
 * return a handle.  Header flags (offset 36): bit 0 = tied head; bit 1 = the paper's own block
 * (Alg. 1 l.4; R#23): every layer is followed by u <- LayerNorm(W2 GELU(W1 u + b1) + b2)
 * with hidden width d_ff (u32 at offset 40) and the per-layer tensors ffn_w1 [d_ff][D], ffn_b1, ffn_w2
 * [D][d_ff], ffn_b2, ln_w, ln_b after W_out; with bit 0 clear an untied head [256][D] follows the layers.
 * Supported: d_state = 16, d_conv = 4, expand = 2, d_model a multiple of 64 and <= 512, dt_rank a
 * multiple of 4 and <= 64, d_ff a multiple of 64 and <= 4096, fp32 or bf16 matrices; else
 * BOA_E_UNSUPPORTED.  Flag bits beyond 0-1, or bit 1 disagreeing with d_ff > 0: BOA_E_FORMAT.
 * The blob is not referenced after the call returns. */
int boa_model_load(const void* weights, size_t nbytes, boa_model** out);
void boa_model_free(boa_model* m);

/* 64-bit fingerprint stored in every container: (arithmetic word << 32) | CRC-32(blob).
 * Tables are only reproducible with the same weights AND the same arithmetic.  The arithmetic word is the
 * kernel generation number XOR the CRC-32 of the fp32 logits that this build's step kernels produce, on this device, for
 * a fixed 120-byte probe input stepped through this model at boa_model_load: a build whose kernels round differently
 * cannot forget to change it. */
uint64_t boa_model_fingerprint(const boa_model* m);

/* ---- compress ---------------------------------------------------------------------------
 * Split `in[0..n)` into ceil(n/chunk_bytes) chunks ("streams"); stream i is bytes
 * [i*chunk_bytes, min(n,(i+1)*chunk_bytes)).  Byte 0 of a stream is stored raw; for t = 0..len-2 the
 * model is stepped on byte t and byte t+1 is range-coded with the resulting table (len-1 symbols),
 * all streams in lock-step.  Writes a BOA1 container to `out`.
 *   in        host|device pointer, n bytes (may be NULL iff n == 0)
 *   chunk_bytes  >= 1 and <= 2^30 (stream positions and the per-stream payload scratch, 2*chunk_bytes + 8, are
 *             32-bit; boa_decompress rejects a header with a larger value as BOA_E_FORMAT)
 *   out       host|device pointer; *out_len = its capacity on entry, bytes written on return.
 *             boa_compress_bound(n, chunk_bytes) is always enough (f >= 1 with total 2^16 bounds a
 *             symbol at 16 bits: payload <= 2*(len-1) + 4 flush bytes).
 * Errors: BOA_E_ARG, BOA_E_CAPACITY (out too small; nothing useful written), BOA_E_NOMEM, BOA_E_CUDA. */
size_t boa_compress_bound(size_t n, size_t chunk_bytes);
int boa_compress(boa_model* m, const uint8_t* in, size_t n, size_t chunk_bytes,
                 uint8_t* out, size_t* out_len, void* cuda_stream);

/* ---- decompress -------------------------------------------------------------------------
 * boa_decompressed_size: read only the 40-byte header (host|device pointer) and return n.
 * boa_decompress: validate header, index CRC and fingerprint, then decode every stream in
 * lock-step with the same step kernels; a stream that has reached its length is masked out.
 *   out       host|device pointer; *out_len = capacity on entry (>= n), n on return.
 * Errors: BOA_E_FORMAT, BOA_E_CRC, BOA_E_MODEL_MISMATCH, BOA_E_CAPACITY, BOA_E_CORRUPT (a decoder
 * needed bytes past the end of its stream or did not consume its stream exactly; output is then
 * undefined), BOA_E_NOMEM, BOA_E_CUDA. */
int boa_decompressed_size(const uint8_t* in, size_t in_len, size_t* n);
int boa_decompress(boa_model* m, const uint8_t* in, size_t in_len,
                   uint8_t* out, size_t* out_len, void* cuda_stream);

/* ---- one container from several GPUs (chunks are independent) ------------------------
 * The chunks of one input are cut into contiguous ranges, one per GPU (weights replicated, no data-path collective).
 * boa_compress_shard: compress a range given as its own bytes - `in` (host|device) points at the first byte of the range's
 *   first chunk, `n` is the byte length of the range (a multiple of chunk_bytes except for the range that holds the end of
 *   the input) - exactly as boa_compress would, but return the parts instead of a container: the range-coder streams back
 *   to back in `payload` (host|device; *payload_len = capacity on entry - 2*n + 4*ceil(n/chunk_bytes) is always enough -
 *   bytes written on return), the per-chunk sizes in `sizes` and first bytes in `first` (HOST arrays of
 *   ceil(n/chunk_bytes) entries; device pointers: BOA_E_ARG).
 * boa_container_assemble: write ONE BOA1 container (fingerprint = boa_model_fingerprint of the model the parts were
 *   compressed with) for the input of `n` bytes from `n_parts` consecutive parts:
 *   header + first bytes + size index + CRC (built on the host from the HOST arrays first[p], sizes[p] of part_chunks[p]
 *   entries) followed by the payload blocks.  `out` is host|device, *out_len capacity on entry (boa_compress_bound is
 *   enough), bytes written on return.  payload[p] (host|device, payload_len[p] bytes = the sum of the part's sizes, else
 *   BOA_E_FORMAT) is copied to its place; a block that already sits there (payload[p] == out + payload_off[p], e.g.
 *   received there from its GPU) is left alone; `payload` may be NULL (index only: the caller places the blocks at
 *   payload_off[p], an optional HOST array of n_parts + 1 byte offsets into `out`; boa_container_index_bytes(n,
 *   chunk_bytes) = payload_off[0]).  The result is byte-identical to boa_compress of the whole input on one GPU.
 *   With host pointers only it is plain host code (no CUDA call; it also runs on a machine without a GPU).
 * boa_decompress_shard: validate the whole container like boa_decompress (header, index CRC, fingerprint) and decode only
 *   chunks [first_chunk, first_chunk + n_chunks_local) into `out` (host|device; byte 0 of chunk first_chunk at out[0];
 *   *out_len capacity on entry, bytes written on return).  A range beyond the container's chunks: BOA_E_ARG.
 * Errors otherwise those of boa_compress / boa_decompress. */
int boa_compress_shard(boa_model* m, const uint8_t* in, size_t n, size_t chunk_bytes, uint8_t* payload, size_t* payload_len,
                       uint32_t* sizes, uint8_t* first, void* cuda_stream);
size_t boa_container_index_bytes(size_t n, size_t chunk_bytes);
int boa_container_assemble(uint64_t fingerprint, size_t n, size_t chunk_bytes, size_t n_parts, const size_t* part_chunks,
                           const uint8_t* const* first, const uint32_t* const* sizes, const uint8_t* const* payload,
                           const size_t* payload_len, uint8_t* out, size_t* out_len, uint64_t* payload_off, void* cuda_stream);
int boa_decompress_shard(boa_model* m, const uint8_t* in, size_t in_len, size_t first_chunk, size_t n_chunks_local,
                         uint8_t* out, size_t* out_len, void* cuda_stream);

/* ---- streaming front end (PAPER Fig. 2) ------------------------------
 * The input is cut into groups of `group_chunks` chunks; every group is compressed into one complete BOA1
 * container (a shard) exactly as boa_compress would, and the shards are concatenated in `out`.  While the
 * step kernels work on group k, a second CUDA stream pre-loads group k+1 from pinned host memory into the
 * other device lane and brings shard k-1 back ("buffer / compress / pre-load", Fig. 2).
 *   in, out      HOST pointers (device pointers: BOA_E_ARG); out_len = capacity on entry, bytes written on return;
 *                boa_stream_bound(n, chunk_bytes, group_chunks) is always enough
 *   shard_len    NULL, or HOST array receiving the byte length of every shard; *n_shards = its capacity on
 *                entry (BOA_E_CAPACITY if < ceil(n / (chunk_bytes * group_chunks))), the shard count on return
 * boa_stream_decompress walks the concatenated shards (each validated like boa_decompress: header, index
 * CRC, fingerprint) with the same two-lane overlap and writes the original bytes; boa_stream_decompressed_size
 * reads only the headers and size indices (HOST pointer) and returns the total length and the shard count.
 * Errors: those of boa_compress / boa_decompress; BOA_E_FORMAT if the buffer is not a whole number of shards. */
size_t boa_stream_bound(size_t n, size_t chunk_bytes, size_t group_chunks);
int boa_stream_compress(boa_model* m, const uint8_t* in, size_t n, size_t chunk_bytes, size_t group_chunks,
                        uint8_t* out, size_t* out_len, uint64_t* shard_len, size_t* n_shards, void* cuda_stream);
int boa_stream_decompressed_size(const uint8_t* in, size_t in_len, size_t* n, size_t* n_shards);
int boa_stream_decompress(boa_model* m, const uint8_t* in, size_t in_len, uint8_t* out, size_t* out_len,
                          void* cuda_stream);

/* ---- FX1: the deterministic fixed-point pipeline (PAPER "Portability") -----------------
 * The paper proposes INT8 / fixed-point Mamba transformations "with explicitly specified rounding and saturation rules" and
 * deterministic normalisation and softmax, so that a container written on one device decodes on another.
 * DESIGN.md section 11 is that specification (Q12.20 values, INT8 rows with power-of-two scales, round-half-even,
 * saturating stores, table-driven integer exp / sigmoid / softplus, integer RMSNorm, the integer table rule); these entry
 * points run it on the GPU, every step an integer kernel (csrc/fx_kernels.cuh; the contractions on tcgen05.mma kind::i8,
 * csrc/fx_gemm_tc.cuh).  Integer arithmetic has one correct
 * answer: logits, tables and whole containers are bit-identical to the exact-integer oracle's (tests).
 *   boa_fx_model_load   parse a BOAW blob of north_star's block with the tied head (flags == 1; else BOA_E_UNSUPPORTED;
 *                       d_model a multiple of 64 and <= 1024, dt_rank <= 64, at most 64 layers), quantise it as section 11
 *                       says (host), lay the INT8 rows out as tensor-core operand images, copy them to the device
 *   boa_fx_model_fingerprint   ('FX01' << 32) | CRC-32(blob): the arithmetic word is a constant - FX1 containers are
 *                       portable by construction, and are never accepted by a floating-point boa_model (nor vice versa)
 *   boa_fx_compress / boa_fx_decompress   as boa_compress / boa_decompress (same BOA1 container, same pointer and error
 *                       conventions); both directions step one byte at a time
 *   boa_fx_debug_step_dump   test-only: logits[r][256] (int32, Q12.20) and cdf[r][257] of row r = stream * n_steps + step
 *   boa_fx_last_launches     kernels launched by the last compress / decompress call of the handle */
typedef struct boa_fx_model boa_fx_model;
int boa_fx_model_load(const void* weights, size_t nbytes, boa_fx_model** out);
void boa_fx_model_free(boa_fx_model* m);
uint64_t boa_fx_model_fingerprint(const boa_fx_model* m);
int boa_fx_compress(boa_fx_model* m, const uint8_t* in, size_t n, size_t chunk_bytes, uint8_t* out, size_t* out_len,
                    void* cuda_stream);
int boa_fx_decompress(boa_fx_model* m, const uint8_t* in, size_t in_len, uint8_t* out, size_t* out_len, void* cuda_stream);
uint64_t boa_fx_last_launches(const boa_fx_model* m);
int boa_fx_debug_step_dump(boa_fx_model* m, const uint8_t* in, size_t n, size_t chunk_bytes, size_t n_steps, int32_t* logits,
                           uint32_t* cdf, void* cuda_stream);

const char* boa_strerror(int code);
/* "file:line: cudaErrorName" of the last CUDA failure seen by the calling thread ("" if none).  Diagnostic only. */
const char* boa_last_cuda_error(void);

/* ---- measurement hooks ---------------------------------------------------------------------------
 * Kernel classes of the step: the order below is the launch order inside one step. */
enum {
  BOA_K_EMBED = 0,   /* S1  byte embedding of the first step of a wave (later steps: in the coder) */
  BOA_K_INPROJ = 1,  /* S2-S4  RMSNorm + in_proj + causal conv1d + SiLU (tensor cores)             */
  BOA_K_CONVX = 2,   /* S5  x_proj (tensor cores, split over k)                                    */
  BOA_K_SCAN = 3,    /* S6-S8  dt_proj + softplus, selective-SSM recurrence, gate (state streamed) */
  BOA_K_OUTPROJ = 4, /* S9  out_proj + residual (tensor cores)                                     */
  BOA_K_HEAD = 5,    /* S10 tied head (tensor cores)                                               */
  BOA_K_CODER = 6,   /* S11-S14 softmax, table, range coder step; S1 of the next step              */
  BOA_K_FINISH = 7,  /* S15/S16 flush, compaction, init                           */
  /* the paper's block only (Alg. 1 l.4), after out_proj of every layer: */
  BOA_K_FFN1 = 8,    /* hidden = GELU(W1 u + b1) (tensor cores; writes the operand image of FFN2)   */
  BOA_K_FFN2 = 9,    /* v = W2 hidden + b2 (tensor cores)                                          */
  BOA_K_LNORM = 10,  /* u = LayerNorm(v); image and block sums of u^2 for the next contraction     */
  /* step path of north_star's block: the dependent contractions between two scans chained in one launch (tc_gemm.cuh) */
  BOA_K_CHAIN_IN_X = 11,      /* in_proj(0) -> x_proj(0)                      */
  BOA_K_CHAIN_OUT_IN_X = 12,  /* out_proj(l) -> in_proj(l+1) -> x_proj(l+1)   */
  BOA_K_CHAIN_OUT_HEAD = 13,  /* out_proj(L-1) -> head                        */
  BOA_K_COUNT = 14
};
typedef struct boa_profile {
  uint64_t launches_total;            /* kernels launched by the last compress/decompress call       */
  uint64_t steps;                     /* model steps taken (max stream length - 1, summed over waves) */
  uint64_t streams;                   /* streams of the last call                                     */
  uint64_t sampled_launches[BOA_K_COUNT]; /* launches that were bracketed by CUDA events             */
  double sampled_ms[BOA_K_COUNT];     /* summed event time of those launches                          */
  double total_ms;                    /* CUDA-event time of the whole call's device work              */
} boa_profile;
/* sample_every = k > 0: every k-th graph batch of the step loop is replaced by one eagerly launched
 * batch whose kernels are individually bracketed by CUDA events on the call's stream (same kernels,
 * same order, same results).  0 (default) = no sampling. */
int boa_set_profiling(boa_model* m, int sample_every);
int boa_get_profile(const boa_model* m, boa_profile* out);

/* ---- test-only exports (the four parity checks of BASELINE.json, tests/test_gpu_*.py) -------------
 * boa_debug_step_dump: run the compress-side step pipeline on `in` (device|host pointer) exactly as
 *   boa_compress does and dump, for stream i and step t (t < n_steps <= chunk_bytes-1), row
 *   r = i*n_steps + t of:  logits[r][256] (fp32, S10), probs[r][256] (fp32 softmax, eq. 6),
 *   cdf[r][257] (uint32, eq. 7).  Any of the three output pointers may be NULL.  All streams must be
 *   full length (n a multiple of chunk_bytes).  Output pointers: device|host.
 * boa_debug_quantise: the table rule alone: logits[rows][256] fp32 -> cdf[rows][257].
 * boa_debug_rc_encode / _decode: the range coder alone, one GPU thread per stream, driven by given
 *   tables: cdf[n_streams][len][257], syms[n_streams][len]; payload of stream i is written at
 *   out + i*cap, its size to sizes[i] (BOA_E_CAPACITY if any would exceed cap).  Decode reads the
 *   same layout and writes syms; BOA_E_CORRUPT on overrun / bytes left over. */
/* boa_debug_gemm: the tensor-core contraction kernel alone (S3/S5/S9/S10; tc_gemm.cuh):
 *   C[M][N] = A[M][K] W[N][K]^T, A and C host|device fp32 row-major, W a HOST fp32 matrix that is cut into
 *   `weight_pieces` (1 or 3) bf16 pieces exactly as boa_model_load does; A is cut into its three pieces by the same
 *   device routine the step kernels use.  grid_ctas = 0 launches one persistent CTA per SM as the time slabs do; a small
 *   positive value forces several tiles per CTA (the accumulator double-buffering path).  grid_ctas = -1 runs the
 *   CTA-pair kernel of the step path instead (tc_gemm2.cuh: tcgen05 cta_group::2, 256 x 128 tiles) with one pair per SM
 *   pair; -2k runs it with k pairs (several tiles per pair).  Both kernels must return the same bits.  K % 64 == 0. */
/* boa_debug_set_slab: enabled = 0 makes boa_compress step one byte at a time, exactly as boa_decompress must, instead
 *   of advancing 16 bytes per pass over the stream state; the container bytes must not change (test).
 * boa_debug_set_max_wave: streams > 0 caps the number of streams stepped together (more chunks then run in waves), as
 *   a small free-memory budget would; 0 restores the default.  Results must not depend on it (test). */
int boa_debug_set_slab(boa_model* m, int enabled);
/* boa_debug_set_chain: enabled = 1 chains the dependent contractions of the step path inside one launch (tc::k_gemm_chain,
 *   2L + 2 launches per step) instead of one kernel per contraction (4L + 2, the default: the chained form measured
 *   neutral).  Same bytes either way (test). */
int boa_debug_set_chain(boa_model* m, int enabled);
/* boa_debug_set_persist: waves of at most `max_streams` streams step inside one launch of the persistent step kernel
 *   (step_persist.cuh; 0 = never, i.e. always the graph of one kernel per phase), with `cluster_ctas` CTAs per row tile of
 *   128 streams (1, 2, 4, 8 or 16; 0 = keep).  Same bytes either way (test). */
int boa_debug_set_persist(boa_model* m, size_t max_streams, int cluster_ctas);
/* boa_debug_set_pair_tiles: the step path's contractions run with CTA-pair tiles (tc_gemm2.cuh) when a wave has at least
 *   `min_row_tiles` row tiles of 128 streams (0 = always; default INT_MAX = never: measured slower).
 *   Same bytes either way. */
int boa_debug_set_pair_tiles(boa_model* m, int min_row_tiles);
int boa_debug_set_max_wave(boa_model* m, size_t streams);
int boa_debug_gemm(const float* A, size_t M, size_t K, const float* W, size_t N, int weight_pieces, int grid_ctas,
                   float* C, void* cuda_stream);
int boa_debug_step_dump(boa_model* m, const uint8_t* in, size_t n, size_t chunk_bytes, size_t n_steps,
                        float* logits, float* probs, uint32_t* cdf, void* cuda_stream);
int boa_debug_quantise(const float* logits, size_t rows, uint32_t* cdf, void* cuda_stream);
int boa_debug_rc_encode(const uint32_t* cdf, const uint8_t* syms, size_t n_streams, size_t len,
                        uint8_t* out, size_t cap, uint32_t* sizes, void* cuda_stream);
int boa_debug_rc_decode(const uint32_t* cdf, const uint8_t* in, size_t cap, const uint32_t* sizes,
                        size_t n_streams, size_t len, uint8_t* syms, void* cuda_stream);

/* ---- an entry point that allocates nothing ----------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it).  boa_rc_encode_packed_noalloc runs S13e-S15 (eq. 8-11) on given tables: one GPU thread per stream
 * codes symbols syms[i][0..len) under cdf[i][t][257] (as boa_debug_rc_encode) into a scratch row, the sizes are scanned
 * on the device, and the payloads are packed back to back into `payload` (stream 0 first):
 *   sizes[i]   bytes of stream i;   payload[sum_{j<i} sizes[j] ...]   its bytes;
 *   status[0]  total payload bytes; status[1]  flags: bit 0 = payload_cap too small (streams that would end beyond
 *              it are not written), bit 1 = a stream overflowed its scratch row (its size reads 0; cannot happen for
 *              valid tables, whose cost is below 2.0007 bytes per symbol).
 * The scratch rows, offsets and running totals - what the other entry points keep in a model's cudaMalloc'ed
 * workspace - live in ONE static device array of boa_noalloc_scratch_bytes() = 4 MiB that every GPU loading the
 * library holds until exit.  The call makes no cudaMalloc / cudaFree / allocating library call and does not
 * synchronise: it enqueues five kernels on `cuda_stream` (used as it is, unlike the calls above) and returns; read
 * sizes / status / payload after synchronising that stream.
 * ALL pointers are DEVICE pointers (staging a host buffer would need an allocation): a host pointer -> BOA_E_ARG.
 * Limit: 256 + 8 n_streams (rounded up to 256) + n_streams * round_up(2 len + 8, 16) <= 4 MiB and n_streams <= 65,536,
 * i.e. n_streams <= boa_noalloc_max_streams(len) (e.g. 255 streams of 8,192 symbols, 7,824 of 256); beyond it
 * BOA_E_CAPACITY, with the numbers in boa_last_cuda_error().  len >= 2^30: the limit is 0.
 * Every call shares the array, which keeps the last call's contents: the call clears the words that must start at
 * zero itself, but calls that OVERLAP on the GPU (different streams, different host threads) race - serialise them. */
size_t boa_noalloc_scratch_bytes(void);
size_t boa_noalloc_max_streams(size_t len);
int boa_rc_encode_packed_noalloc(const uint32_t* cdf, const uint8_t* syms, size_t n_streams, size_t len, uint8_t* payload,
                                 size_t payload_cap, uint32_t* sizes, uint64_t* status, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* BOA_H_ */
