// container.h — host-side BOA1 container header / index and BOAW blob header (no device code).
//
// BOA1 (first byte of each stream, the compressed streams, nominal chunk length, length of the
// final chunk, total uncompressed length, a compact model fingerprint, CRC-protected index):
//     0   'BOA1'            4   u32 version = 1        8   u64 n (uncompressed bytes)
//     16  u32 chunk_bytes   20  u32 last_chunk_len     24  u32 n_chunks
//     28  u32 freq_bits=16  32  u64 model fingerprint
//     40  u8  first[n_chunks], zero-padded to a multiple of 4
//     ..  u32 size[n_chunks]
//     ..  u32 CRC-32 (IEEE 802.3, reflected, as zlib) of every byte before it
//     ..  payload: the n_chunks range-coder streams back to back
#pragma once
#include <stddef.h>
#include <stdint.h>
#include <string.h>

namespace boa {

constexpr size_t kHeaderBytes = 40;
constexpr uint32_t kContainerVersion = 1;
constexpr size_t kMaxChunkBytes = (size_t)1 << 30;   // encoder and decoder limit (per-stream scratch and positions are 32-bit)

struct Crc32Table {
  uint32_t v[256];
  constexpr Crc32Table() : v{} {
    for (uint32_t i = 0; i < 256; ++i) {
      uint32_t c = i;
      for (int k = 0; k < 8; ++k) c = (c & 1u) ? (0xEDB88320u ^ (c >> 1)) : (c >> 1);
      v[i] = c;
    }
  }
};

// built at compile time: different handles may run on different threads (boa.h)
inline uint32_t crc32_ieee(const uint8_t* p, size_t n, uint32_t crc = 0) {
  static constexpr Crc32Table table{};
  crc = ~crc;
  for (size_t i = 0; i < n; ++i) crc = table.v[(crc ^ p[i]) & 0xFFu] ^ (crc >> 8);
  return ~crc;
}

inline uint64_t n_chunks_of(uint64_t n, uint64_t chunk_bytes) { return n ? (n + chunk_bytes - 1) / chunk_bytes : 0; }
inline size_t first_padded(uint64_t nc) { return (size_t)((nc + 3) / 4 * 4); }
inline size_t index_bytes(uint64_t nc) { return kHeaderBytes + first_padded(nc) + 4 * (size_t)nc + 4; }

struct Header {
  uint64_t n;
  uint32_t chunk_bytes, last_len, n_chunks, freq_bits;
  uint64_t fingerprint;
};

inline void put_u32(uint8_t* p, uint32_t v) { for (int i = 0; i < 4; ++i) p[i] = (uint8_t)(v >> (8 * i)); }
inline void put_u64(uint8_t* p, uint64_t v) { for (int i = 0; i < 8; ++i) p[i] = (uint8_t)(v >> (8 * i)); }
inline uint32_t get_u32(const uint8_t* p) { uint32_t v = 0; for (int i = 0; i < 4; ++i) v |= (uint32_t)p[i] << (8 * i); return v; }
inline uint64_t get_u64(const uint8_t* p) { uint64_t v = 0; for (int i = 0; i < 8; ++i) v |= (uint64_t)p[i] << (8 * i); return v; }

inline void write_header(uint8_t* p, const Header& h) {
  memcpy(p, "BOA1", 4);
  put_u32(p + 4, kContainerVersion);
  put_u64(p + 8, h.n);
  put_u32(p + 16, h.chunk_bytes);
  put_u32(p + 20, h.last_len);
  put_u32(p + 24, h.n_chunks);
  put_u32(p + 28, h.freq_bits);
  put_u64(p + 32, h.fingerprint);
}

// returns false on bad magic / version / freq_bits / inconsistent lengths
inline bool parse_header(const uint8_t* p, Header& h) {
  if (memcmp(p, "BOA1", 4) != 0 || get_u32(p + 4) != kContainerVersion) return false;
  h.n = get_u64(p + 8);
  h.chunk_bytes = get_u32(p + 16);
  h.last_len = get_u32(p + 20);
  h.n_chunks = get_u32(p + 24);
  h.freq_bits = get_u32(p + 28);
  h.fingerprint = get_u64(p + 32);
  if (h.freq_bits != 16 || h.chunk_bytes == 0 || h.chunk_bytes > kMaxChunkBytes) return false;
  const uint64_t nc = n_chunks_of(h.n, h.chunk_bytes);
  if (nc != h.n_chunks) return false;
  if (nc ? (h.last_len != h.n - (nc - 1) * (uint64_t)h.chunk_bytes) : (h.last_len != 0)) return false;
  return true;
}

}  // namespace boa
