"""Test-only assembler of ACX-B200 archives from explicit commands, written from FORMAT.md alone.

It contains its own pure-Python rANS *encoder* (FORMAT.md §1.5, encoder paragraph) so that the oracle's decoder is
pinned against something that is neither the oracle nor the C++ encoder.  Used for hand-built archives whose
expected output is written by hand in the tests."""
import struct

M_BITS = 11
M = 1 << M_BITS
MAGIC = bytes([0x41, 0x43, 0x58, 0x42, 0x32, 0x30, 0x30, 0x00])


def normalise(hist):
    """256 counts -> 256 frequencies summing to M, every present symbol >= 1."""
    total = sum(hist)
    if total == 0:
        return [M] + [0] * 255
    f = [max(1, (h * M) // total) if h else 0 for h in hist]
    while sum(f) != M:
        i = max(range(256), key=lambda s: f[s])
        f[i] += 1 if sum(f) < M else -1
    return f


def rans_encode(symbols, tids, freqs):
    """symbols[i] coded with table tids[i] on state i % 32.  Returns (32 initial decoder states, 32 lists of u16 words:
    state k's own stream in the order the decoder consumes it)."""
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
        assert f > 0, "symbol with zero frequency"
        s = i % 32
        if x[s] >= (f << (32 - M_BITS)):
            streams[s].append(x[s] & 0xFFFF)
            x[s] >>= 16
        x[s] = ((x[s] // f) << M_BITS) + (x[s] % f) + c
        assert (1 << 16) <= x[s] < (1 << 32)
    for st in streams:
        st.reverse()
    return x, streams


def build(blocks, N, log2_bs, min_match=4, W=4, levels=None, raw_planes=(0, 1), with_fnv=False, expected=None,
          mutate=None):
    """blocks: list (one per block) of command lists; a command is (literal_bytes, match) with match = (src, length)
    or None (only allowed for the last command of a block).  Returns the archive bytes."""
    n_tables = 3 + W
    BS = 1 << log2_bs
    assert len(blocks) == (N + BS - 1) // BS
    levels = levels or [0] * len(blocks)
    per = []
    hist = [[0] * 256 for _ in range(n_tables)]
    for cmds in blocks:
        cmd, mlen, lit, off, ext_c, ext_m = [], [], bytearray(), [], [], []
        for k, (lb, m) in enumerate(cmds):
            lb = bytes(lb)
            if len(lb) < 255:
                cmd.append(len(lb))
            else:
                cmd.append(255)
                ext_c.append(len(lb) - 255)
            lit += lb
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
        per.append((cmd, mlen, bytes(lit), off, ext_c + ext_m))
        for v in cmd:
            hist[0][v] += 1
        for v in mlen:
            hist[1][v] += 1
        for v in off:
            for p in range(W):
                hist[2 + p][(v >> (8 * p)) & 0xFF] += 1
        for v in lit:
            hist[2 + W][v] += 1
    modes = [0] * n_tables
    for p in raw_planes:
        modes[2 + p] = 1
    freqs = [normalise(h) if modes[t] == 0 else [0] * 256 for t, h in enumerate(hist)]
    payloads, dirs = [], []
    for (cmd, mlen, lit, off, ext) in per:
        syms, tids = list(cmd), [0] * len(cmd)
        syms += mlen
        tids += [1] * len(mlen)
        for p in range(W - 1, -1, -1):
            if modes[2 + p] == 0:
                syms += [(v >> (8 * p)) & 0xFF for v in off]
                tids += [2 + p] * len(off)
        syms += list(lit)
        tids += [2 + W] * len(lit)
        states, streams = rans_encode(syms, tids, freqs)
        words = [w for st in streams for w in st]
        pl, woff = b"", 0
        for k in range(32):                                   # head: (initial state, word_off) per state
            pl += struct.pack("<II", states[k], woff)
            woff += len(streams[k])
        pl += b"".join(struct.pack("<H", w) for w in words)
        pl += b"\0" * (-len(pl) % 4)
        pl += b"".join(struct.pack("<I", e) for e in ext)
        for p in range(W):
            if modes[2 + p] == 1:
                pl += bytes((v >> (8 * p)) & 0xFF for v in off)
        pl += b"\0" * (-len(pl) % 16)
        payloads.append(pl)
        dirs.append((len(cmd), len(mlen), len(lit), len(words), len(ext)))
    tables_off = 160
    dir_off = tables_off + 528 * n_tables
    fnv_off = dir_off + 32 * len(blocks)
    payload_off = fnv_off + (8 * len(blocks) if with_fnv else 0)
    payload_off += -payload_off % 16
    total = payload_off + sum(len(p) for p in payloads)
    tot_lit = sum(d[2] for d in dirs)
    hdr = MAGIC + struct.pack("<IIQQIIIIIIIIQQQQQQQQQQQQ", 2, 160, N, len(blocks), log2_bs, min_match, W, M_BITS, n_tables,
                              max(levels) if levels else 0, max([d[0] for d in dirs] or [0]), 1 if with_fnv else 0,
                              tables_off, dir_off, fnv_off if with_fnv else 0, payload_off, total, tot_lit, N - tot_lit,
                              sum(d[1] for d in dirs), sum(d[0] for d in dirs), 0, 0, 0)
    assert len(hdr) == 160
    out = bytearray(hdr)
    for t in range(n_tables):
        out += struct.pack("<IIQ", modes[t], 0, 0) + b"".join(struct.pack("<H", f) for f in freqs[t])
    po = payload_off
    for b, d in enumerate(dirs):
        out += struct.pack("<QIIIIIHH", po, d[0], d[1], d[2], d[3], d[4], levels[b], 0)
        po += len(payloads[b])
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
    assert len(out) == total
    if mutate:
        mutate(out)
    return bytes(out)


def lz_reference(cmds_per_block, N, log2_bs):
    """Independent byte-serial LZ77 reference (FORMAT.md §2) on explicit commands."""
    out = bytearray(N)
    BS = 1 << log2_bs
    for b, cmds in enumerate(cmds_per_block):
        dst = b * BS
        for lb, m in cmds:
            out[dst:dst + len(lb)] = lb
            dst += len(lb)
            if m is not None:
                src, ln = m
                for i in range(ln):
                    out[dst + i] = out[src + i]
                dst += ln
    return bytes(out)
