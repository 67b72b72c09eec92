// TEST-ONLY host emulator + hazard checker for the work list (never on the product path).
//
// It runs the product's own unit decode (paper_2606_26607_b200/csrc/moebius_units.h: decode_box,
// box_chunk, tp_src_rank, seg_boxes) over HOST copies of the unified buffer and the staging
// buffer, unit by unit in list order, and checks every 16-byte access against the ordering the
// wait/signal counters guarantee on the device:
//   write after read  (WAR): the reading segment must be ordered before the writing one;
//   read after write  (RAW): the writing segment must be ordered before the reading one;
//   write after write (WAW): ordered likewise.  Same-segment conflicts are always violations
// (units of one segment run concurrently).  This is the planner's unit test.
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <vector>

#include "../../paper_2606_26607_b200/csrc/moebius_units.h"

using namespace moebius;

namespace {

struct Checker {
  char* base; int64_t base_bytes; char* stg; int64_t stg_bytes;
  std::vector<int32_t> rd, wr;          // per 16-byte chunk: last reading / writing segment, -1 none
  std::vector<uint8_t> before;          // before[a*n+b] = 1: segment a completes before b starts
  int n; int64_t violations; int64_t oob; int64_t bytes_read, bytes_written;
  int64_t chunk_of(const char* p) const {
    if (p >= base && p + 16 <= base + base_bytes) return (p - base) >> 4;
    if (stg && p >= stg && p + 16 <= stg + stg_bytes) return (base_bytes >> 4) + ((p - stg) >> 4);
    return -1;
  }
  bool ordered(int a, int b) const { return a != b && before[(size_t)a * n + b]; }
  void on_read(const char* p, int seg, int bytes) {
    for (int o = 0; o < bytes; o += 16) {
      int64_t c = chunk_of(p + o);
      if (c < 0) { ++oob; continue; }
      if (wr[c] >= 0 && !ordered(wr[c], seg)) ++violations;  // RAW not ordered
      rd[c] = seg;
      bytes_read += 16;
    }
  }
  void on_write(const char* p, int seg, int bytes) {
    for (int o = 0; o < bytes; o += 16) {
      int64_t c = chunk_of(p + o);
      if (c < 0) { ++oob; continue; }
      if (rd[c] >= 0 && !ordered(rd[c], seg)) ++violations;  // WAR not ordered
      if (wr[c] >= 0 && !ordered(wr[c], seg)) ++violations;  // WAW not ordered
      wr[c] = seg;
      bytes_written += 16;
    }
  }
};

}  // namespace

extern "C" __attribute__((visibility("default")))
int emul_run(char* base, int64_t base_bytes, char* stg, int64_t stg_bytes, const Seg* segs, int n_segs,
             const KvDesc* kv, const C2dDesc* c2d, int64_t rank_stride, int64_t* out /*[8]*/, const BulkDesc* bulk,
             const WBlk* wblk, int64_t wstg_off) {
  Checker ck;
  ck.base = base; ck.base_bytes = base_bytes; ck.stg = stg; ck.stg_bytes = stg_bytes;
  ck.n = n_segs; ck.violations = ck.oob = ck.bytes_read = ck.bytes_written = 0;
  ck.rd.assign((size_t)((base_bytes + stg_bytes) >> 4), -1);
  ck.wr.assign((size_t)((base_bytes + stg_bytes) >> 4), -1);
  // ordering closure: b waits on counter c with target t == all units signalling c  =>  every
  // segment signalling c is before b, and so is everything before those.
  ck.before.assign((size_t)n_segs * n_segs, 0);
  int64_t bad_wait = 0;
  for (int b = 0; b < n_segs; ++b) {
    if (segs[b].wait_ctr < 0) continue;
    uint64_t tot = 0;
    for (int a = 0; a < n_segs; ++a) if (segs[a].signal_ctr == segs[b].wait_ctr) tot += segs[a].n_units;
    if (tot != segs[b].wait_target) { ++bad_wait; continue; }
    for (int a = 0; a < n_segs; ++a) {
      if (segs[a].signal_ctr != segs[b].wait_ctr) continue;
      if (a >= b) { ++bad_wait; continue; }   // dependencies must point backwards in list order
      ck.before[(size_t)a * n_segs + b] = 1;
      for (int z = 0; z < n_segs; ++z) if (ck.before[(size_t)z * n_segs + a]) ck.before[(size_t)z * n_segs + b] = 1;
    }
  }
  DevParams p;
  memset(&p, 0, sizeof(p));
  p.base = base; p.stg = stg; p.segs = segs; p.kv = kv; p.c2d = c2d; p.bulk = bulk; p.wblk = wblk; p.wstg_off = wstg_off;
  p.rank_stride = rank_stride; p.n_segs = (uint32_t)n_segs;
  uint64_t expect_begin = 0;
  int64_t bad_begin = 0;
  for (int si = 0; si < n_segs; ++si) {
    const Seg& s = segs[si];
    if (s.unit_begin != expect_begin) ++bad_begin;
    expect_begin += s.n_units;
    for (uint32_t u = 0; u < s.n_units; ++u) {
      if (seg_kind(s) == SEG_COPY2D) {
        const C2dDesc& d = c2d[s.desc_begin + u];
        for (uint32_t r = 0; r < d.rows; ++r) {
          // scales are 4-byte granular: account at 16-byte chunk level only for bounds, copy bytes
          const char* src = base + d.src_off + (int64_t)r * d.src_stride;
          char* dst = base + d.dst_off + (int64_t)r * d.dst_stride;
          if (d.src_off < 0 || d.dst_off < 0 || src + d.run_bytes > base + base_bytes || dst + d.run_bytes > base + base_bytes) { ++ck.oob; continue; }
          memmove(dst, src, d.run_bytes);
          ck.bytes_read += d.run_bytes; ck.bytes_written += d.run_bytes;
        }
        continue;
      }
      if (seg_kind(s) == SEG_BULK) {
        BulkUnit bu;
        decode_bulk(s, p, u, bu);
        for (uint32_t t = 0; t < bu.nrows; ++t) {
          const char* src = bu.src + (int64_t)t * bu.src_stride;
          char* dst = bu.dst + (int64_t)t * bu.dst_stride;
          ck.on_read(src, si, (int)bu.piece);
          ck.on_write(dst, si, (int)bu.piece);
          if (ck.chunk_of(src) >= 0 && ck.chunk_of(dst) >= 0 && ck.chunk_of(src + bu.piece - 16) >= 0 && ck.chunk_of(dst + bu.piece - 16) >= 0)
            memmove(dst, src, bu.piece);
        }
        continue;
      }
      uint32_t nb = seg_boxes(s, u);
      for (uint32_t k = 0; k < nb; ++k) {
        Box b;
        decode_box(s, p, u, k, b);
        if (b.lin) {
          if (seg_path(s) == PATH_TMA) {
            // the device moves the WHOLE page image through the tensor maps: rows past the valid
            // tokens are read and written too (unspecified bytes, reading A10)
            ck.on_read(b.lin_src, si, (int)s.ep_page_bytes);
            ck.on_write(b.lin_dst, si, (int)s.ep_page_bytes);
            ck.bytes_read -= s.ep_page_bytes - b.lin_bytes;
            ck.bytes_written -= s.ep_page_bytes - b.lin_bytes;
            if (ck.chunk_of(b.lin_src) >= 0 && ck.chunk_of(b.lin_dst) >= 0 &&
                ck.chunk_of(b.lin_src + s.ep_page_bytes - 16) >= 0 && ck.chunk_of(b.lin_dst + s.ep_page_bytes - 16) >= 0)
              memmove(b.lin_dst, b.lin_src, s.ep_page_bytes);
            continue;
          }
          ck.on_read(b.lin_src, si, (int)b.lin_bytes);
          ck.on_write(b.lin_dst, si, (int)b.lin_bytes);
          if (ck.chunk_of(b.lin_src) >= 0 && ck.chunk_of(b.lin_dst) >= 0 &&
              ck.chunk_of(b.lin_src + b.lin_bytes - 16) >= 0 && ck.chunk_of(b.lin_dst + b.lin_bytes - 16) >= 0)
            memmove(b.lin_dst, b.lin_src, b.lin_bytes);
          continue;
        }
        uint32_t n = b.nrows * b.J * b.cc;
        // like the device: all loads of a box complete before... no -- the device interleaves loads
        // and stores of one box, so a box must not overlap itself either: check chunk by chunk
        for (uint32_t idx = 0; idx < n; ++idx) {
          char *ep, *tp; uint32_t g;
          box_chunk(b, idx, ep, tp, g);
          if (s.ep_is_src) {
            ck.on_read(ep, si, 16);
            for (uint32_t r = 0; r < b.rep; ++r) {
              char* dst = tp + (int64_t)(g * b.rep + r) * rank_stride;
              ck.on_write(dst, si, 16);
              if (ck.chunk_of(ep) >= 0 && ck.chunk_of(dst) >= 0) memcpy(dst, ep, 16);
            }
          } else {
            char* src = tp + (int64_t)tp_src_rank(g, b.rep, b.owner) * rank_stride;
            ck.on_read(src, si, 16);
            ck.on_write(ep, si, 16);
            if (ck.chunk_of(ep) >= 0 && ck.chunk_of(src) >= 0) memcpy(ep, src, 16);
          }
        }
        // PATH_TMA, TP->EP page move: the tensor-map store writes the WHOLE EP page box, so the
        // slots past the valid tokens receive unspecified bytes (reading A10)
        if (seg_path(s) == PATH_TMA && seg_kind(s) == SEG_KV && !s.ep_is_src) {
          uint32_t row_bytes = s.n_groups * s.run_bytes;
          uint32_t pg = s.ep_page_bytes / row_bytes;
          for (uint32_t t = b.nrows; t < pg; ++t) {
            char* row = b.ep + (int64_t)t * row_bytes;
            ck.on_write(row, si, (int)row_bytes);
            if (ck.chunk_of(row) >= 0 && ck.chunk_of(row + row_bytes - 16) >= 0) memset(row, 0xEE, row_bytes);
            ck.bytes_written -= row_bytes;   // not part of the accounted (valid-token) bytes
          }
        }
      }
    }
  }
  out[0] = ck.violations; out[1] = ck.oob; out[2] = bad_wait; out[3] = bad_begin;
  out[4] = ck.bytes_read; out[5] = ck.bytes_written; out[6] = (int64_t)expect_begin; out[7] = 0;
  return 0;
}
