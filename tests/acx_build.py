"""Test-only assembler of ACX-B200 archives (version 3) from explicit commands, written from FORMAT.md alone.

It contains its own pure-Python rANS *encoder* (FORMAT.md §1.7, encoder paragraph) so that the oracle's decoder is
pinned against something that is neither the oracle nor the C++ encoder.  Used for hand-built archives whose
expected output is written by hand in the tests."""
import struct

M_BITS = 11
M = 1 << M_BITS
MQ_BITS = 12
MAGIC = bytes([0x41, 0x43, 0x58, 0x42, 0x32, 0x30, 0x30, 0x00])
TAIL_PAD = 128


def normalise(hist, bits=M_BITS):
    """counts -> frequencies summing to 2^bits, every present symbol >= 1."""
    total, m = sum(hist), 1 << bits
    if total == 0:
        return [m] + [0] * (len(hist) - 1)
    f = [max(1, (h * m) // total) if h else 0 for h in hist]
    while sum(f) != m:
        i = max(range(len(f)), key=lambda s: f[s])
        f[i] += 1 if sum(f) < m else -1
    return f


def rans_encode(symbols, tids, freqs, bits=None):
    """symbols[i] (an index into table tids[i]) coded on state i % 32; bits[t] = precision of table t (default 11).
    Returns (32 initial decoder states, 32 lists of u16 words: state k's own stream in the order the decoder consumes it)."""
    bits = bits or [M_BITS] * len(freqs)
    cums = []
    for f in freqs:
        c = [0]
        for v in f:
            c.append(c[-1] + v)
        cums.append(c)
    x = [1 << 16] * 32
    streams = [[] for _ in range(32)]
    for i in range(len(symbols) - 1, -1, -1):
        f = freqs[tids[i]][symbols[i]]
        c = cums[tids[i]][symbols[i]]
        pb = bits[tids[i]]
        assert f > 0, "symbol with zero frequency"
        s = i % 32
        if x[s] >= (f << (32 - pb)):
            streams[s].append(x[s] & 0xFFFF)
            x[s] >>= 16
        x[s] = ((x[s] // f) << pb) + (x[s] % f) + c
        assert (1 << 16) <= x[s] < (1 << 32)
    for st in streams:
        st.reverse()
    return x, streams


def _segments_of(block):
    """A block is a command list (one segment) or a list of command lists (its segments)."""
    if block and isinstance(block[0], list):
        return block
    return [block]


def build(blocks, N, log2_bs, min_match=4, W=4, levels=None, raw_planes=(0, 1), with_fnv=False, expected=None,
          mutate=None, log2_seg=None, q_min=0, q_mode=0, filler=0x21, seg_levels=None):
    """blocks: list (one per block); a block is a list of commands (one segment) or a list of segments (lists of commands);
    a command is (literal_bytes, match) with match = (src, length) or None (only allowed for the last command of a
    segment).  filler: the byte put into the half of a LITQ pair that lies outside its run (pair mode).  seg_levels:
    overrides the level copies in the segment directory (to build inconsistent archives).  Returns the archive bytes."""
    n_tables = 4 + W
    BS = 1 << log2_bs
    log2_seg = min(log2_bs, 14) if log2_seg is None else log2_seg
    assert len(blocks) == (N + BS - 1) // BS
    levels = levels or [0] * len(blocks)
    per, first_seg = [], []
    hist = [[0] * 256 for _ in range(n_tables)]
    pair_hist = {}
    for b, block in enumerate(blocks):
        first_seg.append(len(per))
        pos = b * BS
        for cmds in _segments_of(block):
            out_start = pos
            cmd, mlen, lit_a, lit_q, q_syms, off, ext_c, ext_m = [], [], bytearray(), bytearray(), [], [], [], []
            for k, (lb, m) in enumerate(cmds):
                lb = bytes(lb)
                if len(lb) < 255:
                    cmd.append(len(lb))
                else:
                    cmd.append(255)
                    ext_c.append(len(lb) - 255)
                if q_min and len(lb) >= q_min:
                    lit_q += lb
                    if q_mode == 1:       # pairs k = pos // 2 .. (pos + L - 1) // 2; the halves outside the run are fillers
                        for kk in range(pos // 2, (pos + len(lb) - 1) // 2 + 1):
                            v0 = lb[2 * kk - pos] if 2 * kk >= pos else filler
                            v1 = lb[2 * kk + 1 - pos] if 2 * kk + 1 < pos + len(lb) else filler
                            q_syms.append(v0 | v1 << 8)
                    else:
                        q_syms += list(lb)
                else:
                    lit_a += lb
                pos += len(lb)
                if m is None:
                    assert k == len(cmds) - 1
                else:
                    src, ln = m
                    t = ln - min_match
                    assert t >= 0
                    if t < 255:
                        mlen.append(t)
                    else:
                        mlen.append(255)
                        ext_m.append(t - 255)
                    off.append(src)
                    pos += ln
            per.append(dict(out_start=out_start, cmd=cmd, mlen=mlen, lit_a=bytes(lit_a), lit_q=bytes(lit_q), q_syms=q_syms,
                            off=off, ext=ext_c + ext_m, level=levels[b]))
            for v in cmd:
                hist[0][v] += 1
            for v in mlen:
                hist[1][v] += 1
            for v in off:
                for p in range(W):
                    hist[2 + p][(v >> (8 * p)) & 0xFF] += 1
            for v in lit_a:
                hist[2 + W][v] += 1
            for v in q_syms:
                if q_mode == 1:
                    pair_hist[v] = pair_hist.get(v, 0) + 1
                else:
                    hist[3 + W][v] += 1
    first_seg.append(len(per))
    modes = [0] * n_tables
    for p in raw_planes:
        modes[2 + p] = 1
    if q_min == 0 or q_mode == 1:
        modes[3 + W] = 2
    freqs = [normalise(h) if modes[t] == 0 else [0] * 256 for t, h in enumerate(hist)]
    # the pair table (FORMAT.md §1.3): entries sorted by pair value; a symbol of LITQ = index of its pair
    qpairs = sorted(pair_hist)
    if q_mode == 1 and not qpairs:
        qpairs, pair_hist = [0], {0: 1}
    qfreq = normalise([pair_hist[v] for v in qpairs], MQ_BITS) if q_mode == 1 else []
    qindex = {v: i for i, v in enumerate(qpairs)}
    all_freqs = freqs + [qfreq]
    all_bits = [M_BITS] * n_tables + [MQ_BITS]
    q_table = n_tables if q_mode == 1 else 3 + W
    payloads, dirs = [], []
    for sg in per:
        cmd, mlen, off = sg["cmd"], sg["mlen"], sg["off"]
        syms, tids = list(cmd), [0] * len(cmd)
        syms += mlen
        tids += [1] * len(mlen)
        for p in range(W - 1, -1, -1):
            if modes[2 + p] == 0:
                syms += [(v >> (8 * p)) & 0xFF for v in off]
                tids += [2 + p] * len(off)
        syms += list(sg["lit_a"])
        tids += [2 + W] * len(sg["lit_a"])
        syms += [qindex[v] for v in sg["q_syms"]] if q_mode == 1 else sg["q_syms"]
        tids += [q_table] * len(sg["q_syms"])
        states, streams = rans_encode(syms, tids, all_freqs, all_bits)
        words = [w for st in streams for w in st]
        pl, woff = b"", 0
        for k in range(32):                                   # head: (initial state, word_off) per state
            pl += struct.pack("<II", states[k], woff)
            woff += len(streams[k])
        pl += b"".join(struct.pack("<H", w) for w in words)
        pl += b"\0" * (-len(pl) % 4)
        pl += b"".join(struct.pack("<I", e) for e in sg["ext"])
        for p in range(W):
            if modes[2 + p] == 1:
                pl += bytes((v >> (8 * p)) & 0xFF for v in off)
        pl += b"\0" * (-len(pl) % 16)
        payloads.append(pl)
        dirs.append((sg["out_start"], len(cmd), len(mlen), len(sg["lit_a"]), len(sg["lit_q"]), len(sg["q_syms"]), len(words),
                     len(sg["ext"]), sg["level"]))
    n_segs = len(per)

    def al(v):
        return v + (-v % 16)
    tables_off = 192
    qtab_off = tables_off + 528 * n_tables
    blocktab_off = al(qtab_off + 4 * len(qfreq))
    dir_off = al(blocktab_off + 8 * (len(blocks) + 1))
    fnv_off = dir_off + 32 * n_segs
    payload_off = al(fnv_off + (8 * len(blocks) if with_fnv else 0))
    total = payload_off + sum(len(p) for p in payloads) + TAIL_PAD
    tot_lit = sum(d[3] + d[4] for d in dirs)
    hdr = MAGIC + struct.pack("<IIQQQ" + "I" * 12 + "Q" * 13, 3, 192, N, len(blocks), n_segs, log2_bs, min_match, W, M_BITS,
                              n_tables, max(levels) if levels else 0, max([d[1] for d in dirs] or [0]), 1 if with_fnv else 0,
                              log2_seg, q_min, q_mode, len(qfreq),
                              tables_off, qtab_off, blocktab_off, dir_off, fnv_off if with_fnv else 0, payload_off, total,
                              tot_lit, N - tot_lit, sum(d[2] for d in dirs), sum(d[1] for d in dirs), sum(d[4] for d in dirs), 0)
    assert len(hdr) == 192
    out = bytearray(hdr)
    for t in range(n_tables):
        out += struct.pack("<IIQ", modes[t], 0, 0) + b"".join(struct.pack("<H", f) for f in freqs[t])
    for v, f in zip(qpairs if q_mode == 1 else [], qfreq):
        out += struct.pack("<HH", v, f)
    out += b"\0" * (blocktab_off - len(out))
    for b in range(len(blocks)):
        out += struct.pack("<IHH", first_seg[b], levels[b], 0)
    out += struct.pack("<IHH", n_segs, 0, 0)
    out += b"\0" * (dir_off - len(out))
    po = payload_off
    for s, d in enumerate(dirs):
        lvl = d[8] if seg_levels is None else seg_levels[s]
        out += struct.pack("<QQHHHHHHHH", po, d[0], d[1], d[2], d[3], d[4], d[5], d[6], d[7], lvl)
        po += len(payloads[s])
    if with_fnv:
        assert expected is not None
        for b in range(len(blocks)):
            h = 0xCBF29CE484222325
            for v in expected[b * BS:(b + 1) * BS]:
                h = ((h ^ v) * 0x100000001B3) & 0xFFFFFFFFFFFFFFFF
            out += struct.pack("<Q", h)
    out += b"\0" * (payload_off - len(out))
    for p in payloads:
        out += p
    out += b"\0" * TAIL_PAD
    assert len(out) == total
    if mutate:
        mutate(out)
    return bytes(out)


def lz_reference(cmds_per_block, N, log2_bs):
    """Independent byte-serial LZ77 reference (FORMAT.md §2) on explicit commands."""
    out = bytearray(N)
    BS = 1 << log2_bs
    for b, block in enumerate(cmds_per_block):
        dst = b * BS
        for cmds in _segments_of(block):
            for lb, m in cmds:
                out[dst:dst + len(lb)] = lb
                dst += len(lb)
                if m is not None:
                    src, ln = m
                    for i in range(ln):
                        out[dst + i] = out[src + i]
                    dst += ln
    return bytes(out)
