// Bitstream container of one coded frame ("J ... and the number of occupied nodes n_d at each level ...
// is encoded in the bitstream as metadata"; L526 "The header stores the number of levels and the node count of each
// level"; L255 per-attribute quantisation steps).  Host-only code: it frames the sections the device calls produce
// (level sizes, quantisation steps, KLT side information, occupancy bytes raw or rANS-coded, leaf weights, RLGR block
// header and streams) into one self-describing, checksummed byte buffer and parses it back without copying.
//
//   file   = header | section table | payloads
//   header = magic "GSNF" | version u16 | n_sections u16 | gsnfs_frame_desc | crc32 of the file (this field zero) | total bytes u64
//   table  = n_sections x { id u32, reserved u32, offset u64 (from the start of the file, 8-byte aligned), bytes u64 }
// All integers little endian (the library only targets little-endian hosts; checked at pack time).
#include <string.h>

#include "gsnfs.h"

namespace {

const uint32_t kMagic = 0x464e5347u;      // "GSNF"
const uint16_t kVersion = 1;

struct FileHeader {
  uint32_t magic;
  uint16_t version;
  uint16_t n_sections;
  gsnfs_frame_desc desc;
  uint32_t crc;
  uint32_t reserved;
  uint64_t total_bytes;
};
struct TableEntry {
  uint32_t id, reserved;
  uint64_t offset, bytes;
};

uint32_t crc32_update(uint32_t crc, const uint8_t* p, uint64_t n) {
  static uint32_t table[256];
  static bool init = false;
  if (!init) {
    for (uint32_t i = 0; i < 256; ++i) {
      uint32_t c = i;
      for (int k = 0; k < 8; ++k) c = (c & 1u) ? 0xedb88320u ^ (c >> 1) : c >> 1;
      table[i] = c;
    }
    init = true;
  }
  crc = ~crc;
  for (uint64_t i = 0; i < n; ++i) crc = table[(crc ^ p[i]) & 0xffu] ^ (crc >> 8);
  return ~crc;
}

uint64_t align8(uint64_t v) { return (v + 7ull) & ~7ull; }

bool little_endian() { const uint32_t one = 1; return *reinterpret_cast<const uint8_t*>(&one) == 1; }

}  // namespace

extern "C" {

uint64_t gsnfs_container_size(const gsnfs_section* sections, int n_sections) {
  if (n_sections < 0 || n_sections > GSNFS_MAX_SECTIONS || (n_sections && !sections)) return 0;
  uint64_t total = align8(sizeof(FileHeader) + sizeof(TableEntry) * (uint64_t)n_sections);
  for (int i = 0; i < n_sections; ++i) total += align8(sections[i].bytes);
  return total;
}

int gsnfs_container_pack(const gsnfs_frame_desc* desc, const gsnfs_section* sections, int n_sections, uint8_t* out,
                         uint64_t capacity, uint64_t* written) {
  if (!desc || !out || !written || n_sections < 0 || n_sections > GSNFS_MAX_SECTIONS || (n_sections && !sections) ||
      !little_endian())
    return GSNFS_E_INVALID_ARGUMENT;
  for (int i = 0; i < n_sections; ++i)
    if (sections[i].bytes && !sections[i].data) return GSNFS_E_INVALID_ARGUMENT;
  const uint64_t total = gsnfs_container_size(sections, n_sections);
  if (total > capacity) return GSNFS_E_CAPACITY;
  FileHeader h;
  memset(&h, 0, sizeof(h));
  h.magic = kMagic; h.version = kVersion; h.n_sections = (uint16_t)n_sections; h.desc = *desc; h.total_bytes = total;
  uint64_t off = align8(sizeof(FileHeader) + sizeof(TableEntry) * (uint64_t)n_sections);
  const uint64_t payload0 = off;
  memset(out, 0, (size_t)payload0);
  TableEntry* tab = reinterpret_cast<TableEntry*>(out + sizeof(FileHeader));
  for (int i = 0; i < n_sections; ++i) {
    tab[i].id = sections[i].id; tab[i].reserved = 0; tab[i].offset = off; tab[i].bytes = sections[i].bytes;
    if (sections[i].bytes) memcpy(out + off, sections[i].data, (size_t)sections[i].bytes);
    const uint64_t pad = align8(sections[i].bytes) - sections[i].bytes;
    if (pad) memset(out + off + sections[i].bytes, 0, (size_t)pad);
    off += align8(sections[i].bytes);
  }
  h.crc = 0;                                                     // the checksum covers the whole file with this field zero
  h.crc = crc32_update(crc32_update(0u, reinterpret_cast<const uint8_t*>(&h), sizeof(h)), out + sizeof(FileHeader),
                       total - sizeof(FileHeader));
  memcpy(out, &h, sizeof(h));
  *written = total;
  return GSNFS_OK;
}

int gsnfs_container_unpack(const uint8_t* buf, uint64_t bytes, gsnfs_frame_desc* desc, gsnfs_section* sections,
                           int max_sections, int* n_sections) {
  if (!buf || !desc || !n_sections || (max_sections && !sections) || !little_endian()) return GSNFS_E_INVALID_ARGUMENT;
  if (bytes < sizeof(FileHeader)) return GSNFS_E_CORRUPT_STREAM;
  FileHeader h;
  memcpy(&h, buf, sizeof(h));
  if (h.magic != kMagic || h.version != kVersion || h.total_bytes > bytes || h.n_sections > GSNFS_MAX_SECTIONS)
    return GSNFS_E_CORRUPT_STREAM;
  const uint64_t tab_end = sizeof(FileHeader) + sizeof(TableEntry) * (uint64_t)h.n_sections;
  if (tab_end > h.total_bytes) return GSNFS_E_CORRUPT_STREAM;
  {
    FileHeader z = h;
    z.crc = 0;
    const uint32_t crc = crc32_update(crc32_update(0u, reinterpret_cast<const uint8_t*>(&z), sizeof(z)),
                                      buf + sizeof(FileHeader), h.total_bytes - sizeof(FileHeader));
    if (crc != h.crc) return GSNFS_E_CORRUPT_STREAM;
  }
  if (h.n_sections > max_sections) return GSNFS_E_CAPACITY;
  const TableEntry* tab = reinterpret_cast<const TableEntry*>(buf + sizeof(FileHeader));
  for (int i = 0; i < h.n_sections; ++i) {
    TableEntry e;
    memcpy(&e, tab + i, sizeof(e));
    if ((e.offset & 7ull) || e.offset < tab_end || e.offset > h.total_bytes || e.bytes > h.total_bytes - e.offset)
      return GSNFS_E_CORRUPT_STREAM;
    sections[i].id = e.id;
    sections[i].data = e.bytes ? buf + e.offset : nullptr;
    sections[i].bytes = e.bytes;
  }
  *desc = h.desc;
  *n_sections = h.n_sections;
  return GSNFS_OK;
}

}  // extern "C"
