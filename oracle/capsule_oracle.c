/*
 * ORACLE — TEST INFRASTRUCTURE ONLY.  Not part of the product path.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, load or call this file.  It shares no code with the CUDA path.
 *
 * Byte-level capsule: snapshot / restore of a closed, named set of contiguous buffers
 * as plain memcpy of each row's valid byte range.
 *
 * Source: PAPER.md:117-129 (Algorithm 1: "cap.bytes <- device-copy of B valid at P'";
 * "copy cap.bytes back into B"), PAPER.md:86 (§3 Definition: a small fixed-size part +
 * a KV region "valid over [0,P)"), PAPER.md:165 (§5 layer (1): "the stored buffers are
 * copied back byte-for-byte").  fork = n restores; rollback = restore
 * of an earlier capsule.
 *
 * Row model (the reading in DESIGN.md "Readings" #15: only the valid range is copied):
 *   a row is n_seg segments, segment s starting at base + s*seg_stride;
 *   the valid bytes of each segment at boundary P are  fixed_bytes + P*bytes_per_token.
 * Slab layout (the contract stated in include/esc.h, restated here independently):
 *   rows in table order; each row starts at the next multiple of 256 bytes; inside a row,
 *   each segment starts at the next multiple of 16 bytes.  Padding bytes are don't-care.
 */
#include <stddef.h>
#include <stdint.h>
#include <string.h>

typedef struct {
    uint8_t* base;
    uint64_t capacity_bytes;
    uint64_t fixed_bytes;
    uint64_t bytes_per_token;
    uint32_t n_seg;
    uint32_t pad_;
    uint64_t seg_stride;
} oracle_row;

static uint64_t up(uint64_t x, uint64_t a) { return (x + a - 1) / a * a; }

static uint64_t seg_valid(const oracle_row* r, uint64_t P) {
    return r->fixed_bytes + P * r->bytes_per_token;
}

/* 0 if every segment's valid range fits its buffer, else -1 */
static int check(const oracle_row* rows, int n, uint64_t P) {
    for (int i = 0; i < n; ++i) {
        const oracle_row* r = &rows[i];
        if (r->n_seg == 0) return -1;
        uint64_t sv = seg_valid(r, P);
        if (r->n_seg > 1 && sv > r->seg_stride) return -1;
        if ((uint64_t)(r->n_seg - 1) * r->seg_stride + sv > r->capacity_bytes) return -1;
    }
    return 0;
}

/* sum of valid bytes over all rows (no padding) */
int64_t esc_oracle_capsule_payload_bytes(const oracle_row* rows, int n, uint64_t P) {
    if (check(rows, n, P)) return -1;
    uint64_t tot = 0;
    for (int i = 0; i < n; ++i) tot += (uint64_t)rows[i].n_seg * seg_valid(&rows[i], P);
    return (int64_t)tot;
}

/* slab bytes needed, padding included */
int64_t esc_oracle_capsule_slab_bytes(const oracle_row* rows, int n, uint64_t P) {
    if (check(rows, n, P)) return -1;
    uint64_t off = 0;
    for (int i = 0; i < n; ++i) {
        off = up(off, 256);
        uint64_t sv = seg_valid(&rows[i], P);
        for (uint32_t s = 0; s < rows[i].n_seg; ++s) { off = up(off, 16); off += sv; }
    }
    return (int64_t)off;
}

/* slab offset of (row, segment); -1 if out of range */
int64_t esc_oracle_capsule_seg_offset(const oracle_row* rows, int n, uint64_t P, int row, uint32_t seg) {
    if (check(rows, n, P) || row < 0 || row >= n || seg >= rows[row].n_seg) return -1;
    uint64_t off = 0;
    for (int i = 0; i < n; ++i) {
        off = up(off, 256);
        uint64_t sv = seg_valid(&rows[i], P);
        for (uint32_t s = 0; s < rows[i].n_seg; ++s) {
            off = up(off, 16);
            if (i == row && s == seg) return (int64_t)off;
            off += sv;
        }
    }
    return -1;
}

static int walk(const oracle_row* rows, int n, uint64_t P, uint8_t* slab, uint64_t slab_bytes, int to_slab) {
    if (check(rows, n, P)) return -1;
    if ((uint64_t)esc_oracle_capsule_slab_bytes(rows, n, P) > slab_bytes) return -2;
    uint64_t off = 0;
    for (int i = 0; i < n; ++i) {
        off = up(off, 256);
        uint64_t sv = seg_valid(&rows[i], P);
        for (uint32_t s = 0; s < rows[i].n_seg; ++s) {
            off = up(off, 16);
            uint8_t* live = rows[i].base + (uint64_t)s * rows[i].seg_stride;
            if (to_slab) memcpy(slab + off, live, sv);
            else         memcpy(live, slab + off, sv);
            off += sv;
        }
    }
    return 0;
}

/* snapshot(P): live rows -> slab */
int esc_oracle_capsule_snapshot(const oracle_row* rows, int n, uint64_t P, uint8_t* slab, uint64_t slab_bytes) {
    return walk(rows, n, P, slab, slab_bytes, 1);
}

/* restore(cap): slab -> live rows; bytes beyond the valid range are untouched */
int esc_oracle_capsule_restore(const oracle_row* rows, int n, uint64_t P, const uint8_t* slab, uint64_t slab_bytes) {
    return walk(rows, n, P, (uint8_t*)slab, slab_bytes, 0);
}

/* P' = floor(P / C) * C   (Algorithm 1; §5) */
uint64_t esc_oracle_align_boundary(uint64_t P, uint64_t C) { return C ? (P / C) * C : P; }
