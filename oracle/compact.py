"""CPU ORACLE of the compact record encodings (second half: "sparse/bit-packed record
encoding (non-empty bins only) to raise the compression ratio"; the paper's "(count, p50, p99)" record of
"approximately 200 triples ... about 2.7 KB") — TEST INFRASTRUCTURE, NOT PRODUCT.
Plain Python + struct, one field after the other in the order DESIGN.md §3 R37 / R38 state; no numpy tricks.
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this; it shares no code with
paper_2606_20374_b200 and imports nothing from it.

Input = the oracle's own dense table (oracle.Oracle.records(): header 64 B | span[P+1] 32 B | cell[S] 160 B).

R37  SPARSE record (lossless), every field little-endian, every part 8-byte aligned:
       header 64 B   as R17, with version = 2, reserved0 = number of non-empty cells (count != 0),
                     reserved1 = byte length of this sparse record
       u64 phase_mask          bit k set iff phase span k (k < P) has n_events != 0; the whole-iteration span
                               lives in the header and is not repeated
       argus_span 32 B         for every set bit, ascending k
       cell entry              for every non-empty cell, ascending sig:
           u32 sig | u8 b0 | u8 nb | u16 0      b0 = bucket(min), nb = bucket(max) - b0 + 1 (R4 buckets)
           u64 count | u64 sum | u64 min | u64 max
           u32 hist[b0 .. b0 + nb)              the only buckets that can be non-zero
           u32 0 when nb is odd                 (pad to 8 bytes)
R38  TRIPLE record (the paper's, lossy: what NEXT-1 keeps of a cell):
       header 64 B   as R17, with version = 3, reserved0 = number of cells with >= 1 cluster, reserved1 = length
       u64 phase_mask + spans  as R37
       cell entry              for every cell with n_clusters > 0, ascending sig:
           u32 sig | u32 n_clusters
           n_clusters x {u32 count | u16 p50_bin | u16 p99_bin}
The records of a table follow each other in (rank, step) order; offsets[k] = first byte of record k,
offsets[R*T] = total length.

Pins (tests/test_oracle_compact.py, -m "not gpu"): tests/golden/compact_handworked.txt — both encodings of the
hand-worked example, every byte derived by hand from the layout above; decoding the sparse stream with an
independent reader gives back the dense table bit for bit (tiny, invalid events included); length formula;
an all-empty table; a cell that reaches bucket 31.
"""
from __future__ import annotations

import struct
from typing import List, Sequence, Tuple

import numpy as np

MAGIC = 0x53475241


def _bucket(d: int) -> int:
    """R4: 0 for d <= 1, else min(31, floor(log2 d))."""
    return 0 if d <= 1 else min(31, d.bit_length() - 1)


def _header_fields(rec: bytes):
    return struct.unpack_from("<IHHIIIIQqqQQ", rec, 0)


def _spans_part(rec: bytes, P: int) -> Tuple[int, List[bytes]]:
    mask, parts = 0, []
    for k in range(P):
        sp = rec[64 + 32 * k: 64 + 32 * (k + 1)]
        n = struct.unpack_from("<Q", sp, 24)[0]
        if n != 0:
            mask |= 1 << k
            parts.append(sp)
    return mask, parts


def sparse_encode(records: np.ndarray, S: int, P: int) -> Tuple[bytes, List[int]]:
    """records: uint8 [n_records][64 + 32 (P+1) + 160 S] (finalised).  Returns (stream, offsets[n_records + 1])."""
    out = bytearray()
    offsets = [0]
    for row in records:
        rec = bytes(row)
        magic, ver, n_ph, n_sg, rank, step, _r0, n_ev, mn, mx, it, _r1 = _header_fields(rec)
        mask, span_parts = _spans_part(rec, P)
        body = bytearray(struct.pack("<Q", mask))
        for sp in span_parts:
            body += sp
        n_cells = 0
        cell0 = 64 + 32 * (P + 1)
        for s in range(S):
            c = rec[cell0 + 160 * s: cell0 + 160 * (s + 1)]
            count, sm, cmin, cmax = struct.unpack_from("<QQQQ", c, 0)
            if count == 0:
                continue
            hist = struct.unpack_from("<32I", c, 32)
            b0 = _bucket(cmin)
            nb = _bucket(cmax) - b0 + 1
            body += struct.pack("<IBBH", s, b0, nb, 0)
            body += struct.pack("<QQQQ", count, sm, cmin, cmax)
            body += struct.pack("<%dI" % nb, *hist[b0:b0 + nb])
            if nb & 1:
                body += struct.pack("<I", 0)
            n_cells += 1
        length = 64 + len(body)
        out += struct.pack("<IHHIIIIQqqQQ", magic, 2, n_ph, n_sg, rank, step, n_cells, n_ev, mn, mx, it, length)
        out += body
        offsets.append(len(out))
    return bytes(out), offsets


def triple_encode(records: np.ndarray, S: int, P: int, clusters: Sequence[Sequence[Sequence[Tuple[int, int, int]]]]
                  ) -> Tuple[bytes, List[int]]:
    """clusters[k][s] = the (count, p50_bin, p99_bin) triples of cell s of record k (NEXT-1's output)."""
    out = bytearray()
    offsets = [0]
    for k, row in enumerate(records):
        rec = bytes(row)
        magic, ver, n_ph, n_sg, rank, step, _r0, n_ev, mn, mx, it, _r1 = _header_fields(rec)
        mask, span_parts = _spans_part(rec, P)
        body = bytearray(struct.pack("<Q", mask))
        for sp in span_parts:
            body += sp
        n_cells = 0
        for s in range(S):
            tr = clusters[k][s]
            if len(tr) == 0:
                continue
            body += struct.pack("<II", s, len(tr))
            for cnt, p50, p99 in tr:
                body += struct.pack("<IHH", cnt, p50, p99)
            n_cells += 1
        length = 64 + len(body)
        out += struct.pack("<IHHIIIIQqqQQ", magic, 3, n_ph, n_sg, rank, step, n_cells, n_ev, mn, mx, it, length)
        out += body
        offsets.append(len(out))
    return bytes(out), offsets
