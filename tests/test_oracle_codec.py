"""Pins for the oracle's stream writer/parser and decoders.

north_star pins: (1) zero-threshold round trip reproduces the input exactly; (2) a constant
light field reduces to the root level; (3) decode(encode(x)) equals the encoder's own
reconstruction; (4) brute-force per-pixel reconstruction on tiny light fields agrees.
A pure-Python reader written from DESIGN.md "Stream format v1" pins the byte layout.
"""
import struct

import numpy as np
import pytest

import oracle as orc
import workloads as wl
from conftest import random_lf


def _encode(lf, h, B=4, W=4, tau_ref=0, tau_res=0, policy=orc.POLICY_ADAPTIVE, bg=(0, 0, 0)):
    V, U, Ht, Ws, _ = lf.shape
    p = orc.make_params(U, V, Ws, Ht, h, B, W, tau_ref, tau_res, policy, background=bg, seed=77)
    data, info, tree = orc.encode(lf, p)
    return data, info, tree


# ---------------------------------------------------------------- pin 1: lossless
@pytest.mark.parametrize("policy", [orc.POLICY_ADAPTIVE, orc.POLICY_ALL, orc.POLICY_LITERAL])
def test_zero_threshold_roundtrip_is_exact(policy):
    rng = np.random.default_rng(0)
    lf = random_lf(rng, 5, 4, 24, 16)
    data, info, tree = _encode(lf, 2, W=5, policy=policy)
    assert np.array_equal(tree.reconstruct(), lf)            # P1
    s = orc.Stream(data)
    assert np.array_equal(s.decode_full(), lf)               # P2
    assert info["psnr"] == float("inf")


def test_cfg1_lossless_roundtrip(enc):
    cfg, lf, data, info, s = enc("cfg1")
    assert np.array_equal(s.decode(wl.all_coords(cfg)).reshape(lf.shape), lf)


# ---------------------------------------------------------------- pin 2: constant LF -> root only
def test_identical_views_reduce_to_root():
    rng = np.random.default_rng(1)
    img = rng.integers(0, 256, (16, 16, 3)).astype(np.uint8)
    lf = np.broadcast_to(img, (4, 4, 16, 16, 3)).copy()
    data, info, tree = _encode(lf, 2, tau_ref=1, tau_res=1)
    s = orc.Stream(data)
    st = s.stats_decode(wl.all_coords(wl.Config("x", 4, 4, 16, 16, 2, 1, 0, 0, None, 0, 16, 16, 1, 0)))
    assert st["payload_bits15"] == 0 and st["mv_bits15"] == 0   # nothing but flags and the root is read
    assert np.array_equal(s.decode_full(), lf)
    # constant colour: the root RKV is that colour everywhere
    lf2 = np.empty((4, 4, 8, 8, 3), dtype=np.uint8)
    lf2[...] = (200, 50, 120)
    data2, _, _ = _encode(lf2, 2, tau_ref=1, tau_res=1)
    assert np.array_equal(orc.Stream(data2).decode_full(), lf2)


def test_huge_thresholds_leave_only_the_rkv_chain():
    # all thresholds huge -> pixel = colour-inverse of the top RKV sample
    rng = np.random.default_rng(2)
    lf = random_lf(rng, 4, 4, 16, 16)
    data, info, tree = _encode(lf, 2, tau_ref=10 ** 6, tau_res=10 ** 6)
    full = orc.Stream(data).decode_full()
    for v in range(4):
        for u in range(4):
            ycc = [tree.plane("X", 2, u >> 2, v >> 2, c).astype(int) for c in range(3)]
            t = ycc[0] - np.floor_divide(ycc[2], 2)
            g = ycc[2] + t
            b = t - np.floor_divide(ycc[1], 2)
            r = b + ycc[1]
            assert np.array_equal(full[v, u], np.clip(np.stack([r, g, b], -1), 0, 255))


# ---------------------------------------------------------------- pin 3: P1 = P2
@pytest.mark.parametrize("name", ["cfg1_lossy", "mini2", "mini3", "mini4", "mini_h8", "mini_w64"])
def test_stream_decode_equals_encoder_reconstruction(enc, name):
    cfg, lf, data, info, s = enc(name)
    assert np.array_equal(s.decode_full(), info["p1"])
    assert 25.0 < info["psnr"] < 60.0


@pytest.mark.parametrize("policy", [orc.POLICY_ADAPTIVE, orc.POLICY_ALL, orc.POLICY_LITERAL])
def test_p1_equals_p2_all_policies_lossy(policy):
    rng = np.random.default_rng(3)
    lf = random_lf(rng, 5, 5, 24, 20)
    data, info, tree = _encode(lf, 2, W=6, tau_ref=25, tau_res=60, policy=policy)
    assert np.array_equal(orc.Stream(data).decode_full(), tree.reconstruct())


# ---------------------------------------------------------------- pin 4: brute force on tiny LFs
def test_brute_force_decoder_agrees_on_tiny_lf():
    rng = np.random.default_rng(4)
    lf = random_lf(rng, 4, 4, 16, 16)
    for tau in (0, 40):
        data, info, tree = _encode(lf, 2, W=2, tau_ref=tau // 2, tau_res=tau)
        s = orc.Stream(data)
        coords = wl.all_coords(wl.Config("x", 4, 4, 16, 16, 2, 1, 0, 0, None, 0, 16, 16, 1, 0))
        sel = coords[rng.permutation(len(coords))[:600]]
        assert np.array_equal(s.decode_brute(sel), s.decode(sel))


# ---------------------------------------------------------------- independent reader of the byte layout
class PyStream:
    """Pure-Python reader/decoder written from DESIGN.md 'Stream format v1' (not from the C code)."""

    def __init__(self, data):
        self.d = data
        assert data[:4] == b"HMLF"
        ver, hb = struct.unpack_from("<HH", data, 4)
        assert (ver, hb) == (1, 160)
        (self.U, self.V, self.Ws, self.Ht, self.h, self.B, self.W, nch, self.tau_ref, self.tau_res) = struct.unpack_from("<10I", data, 8)
        assert nch == 3 and data[48] == 1 and data[49] == 0 and data[50] == 0
        self.geom = struct.unpack_from("<9f", data, 56)
        self.n_pc, = struct.unpack_from("<Q", data, 104)
        self.off_rkv, self.off_dir, self.off_flags, self.off_pay, self.off_mv, self.total = struct.unpack_from("<6Q", data, 112)
        self.nbx, self.nby = self.Ws // self.B, self.Ht // self.B
        self.nblk = self.nbx * self.nby
        self.dims = [((self.U + (1 << L) - 1) >> L, (self.V + (1 << L) - 1) >> L) for L in range(self.h + 1)]
        self.base, k = {}, 0
        for L in range(self.h - 1, -1, -1):
            self.base[L] = k
            k += self.dims[L][0] * self.dims[L][1] * 3
        assert k == self.n_pc

    def bits(self, sec_off, bitpos, n):
        v = 0
        for j in range(n):
            p = bitpos + j
            v |= ((self.d[sec_off + (p >> 3)] >> (p & 7)) & 1) << j
        return v

    @staticmethod
    def layout(N):
        import math
        if N <= 1:
            return 0, 0
        b = math.ceil(math.log2(N))
        mt = max(0, math.ceil(math.log2(N / 3)))
        mq = max(0, math.ceil(math.log2(N / 5)))
        cands = [(15 * b, 0, b), (24 + 15 * mt, 1, mt), (35 + 15 * mq, 2, mq)]
        _, lay, m = min(cands, key=lambda c: (c[0], c[1]))
        return lay, m

    def bise_at(self, sec_off, bitoff, N, i):
        lay, m = self.layout(N)
        if lay == 0:
            return self.bits(sec_off, bitoff + i * m, m)
        G, radix, hb = (5, 3, 8) if lay == 1 else (3, 5, 7)
        g, k = divmod(i, G)
        gb = bitoff + g * (hb + G * m)
        digit = (self.bits(sec_off, gb, hb) // radix ** k) % radix
        return (digit << m) | self.bits(sec_off, gb + hb + k * m, m)

    def dirent(self, L, pu, pv, c):
        k = self.base[L] + (pv * self.dims[L][0] + pu) * 3 + c
        off, N, n_res, n_pred, foff, poff, moff = struct.unpack_from("<iIIIQQQ", self.d, self.off_dir + 48 * k)
        return off, N, foff, poff, moff

    def flag(self, foff, which, b):
        fbytes = ((self.nblk + 31) // 32) * 4
        return (self.d[self.off_flags + foff + which * fbytes + (b >> 3)] >> (b & 7)) & 1

    def rank(self, foff, which, b):
        return sum(self.flag(foff, which, j) for j in range(b))

    def value(self, L, pu, pv, c, x, y):
        off, N, foff, poff, _ = self.dirent(L, pu, pv, c)
        b = (y // self.B) * self.nbx + x // self.B
        if not self.flag(foff, 0, b):
            return 0
        i = self.rank(foff, 0, b) * self.B * self.B + (y % self.B) * self.B + (x % self.B)
        return off + self.bise_at(self.off_pay, poff, N, i)

    def pixel(self, u, v, x, y):
        h, W = self.h, self.W
        n_top = self.dims[h][0] * self.dims[h][1]
        npx = self.Ws * self.Ht
        idx = ((v >> h) * self.dims[h][0] + (u >> h)) * npx + y * self.Ws + x
        acc = [self.d[self.off_rkv + idx]]
        for c in (1, 2):
            acc.append(struct.unpack_from("<h", self.d, self.off_rkv + n_top * npx + (c - 1) * n_top * npx * 2 + idx * 2)[0])
        for c in range(3):
            for L in range(h):
                pu, pv = u >> L, v >> L
                e = self.value(L, pu, pv, c, x, y)
                if (pu | pv) & 1:
                    _, _, foff, _, moff = self.dirent(L, pu, pv, c)
                    b = (y // self.B) * self.nbx + x // self.B
                    if self.flag(foff, 1, b):
                        nd = 2 * W + 1
                        r = self.bise_at(self.off_mv, moff, 2 * nd * nd, self.rank(foff, 1, b))
                        mode, rem = divmod(r, nd * nd)
                        dy, dx = rem // nd - W, rem % nd - W
                        q = 0
                        if 0 <= x + dx < self.Ws and 0 <= y + dy < self.Ht:
                            q = self.value(L, pu & ~1, pv & ~1, c, x + dx, y + dy)
                        e += -q if mode else q
                acc[c] += e
        Y, Co, Cg = acc
        t = Y - (Cg >> 1)
        G = Cg + t
        Bl = t - (Co >> 1)
        R = Bl + Co
        return tuple(min(255, max(0, z)) for z in (R, G, Bl))


@pytest.mark.parametrize("name,n", [("cfg1_lossy", 300), ("mini3", 300), ("mini4", 200)])
def test_python_reader_of_the_documented_format_agrees(enc, name, n):
    cfg, lf, data, info, s = enc(name)
    ps = PyStream(data)
    assert (ps.U, ps.V, ps.Ws, ps.Ht, ps.h, ps.B, ps.W) == (cfg.U, cfg.V, cfg.Ws, cfg.Ht, cfg.height, cfg.block, cfg.window)
    g = wl.geometry(cfg)
    assert np.allclose(ps.geom, [*g["uv_origin"], *g["uv_step"], *g["st_origin"], *g["st_step"], g["z_st"]])
    coords = wl.random_coords(cfg, n)
    expect = s.decode(coords)
    for q, e in zip(coords, expect):
        assert ps.pixel(*map(int, q)) == tuple(e)


# ---------------------------------------------------------------- container behaviour
def test_parse_errors_are_distinct(enc):
    cfg, lf, data, info, s = enc("cfg1_lossy")
    bad = bytearray(data)
    bad[0] ^= 0xFF
    for blob, code in [(bytes(bad), orc.E_MAGIC), (data[:100], orc.E_TRUNCATED), (data[:len(data) - 9], orc.E_TRUNCATED),
                       (data[:4] + b"\x09\x00" + data[6:], orc.E_VERSION), (data[:6], orc.E_TRUNCATED)]:
        with pytest.raises(orc.OracleError) as ei:
            orc.Stream(blob)
        assert ei.value.code == code


def test_header_roundtrip_and_determinism(enc):
    cfg, lf, data, info, s = enc("mini2")
    p = s.params
    assert (p.U, p.V, p.Ws, p.Ht, p.height, p.block, p.window, p.tau_res, p.tau_ref) == (8, 8, 96, 80, 3, 4, 16, 48, 24)
    p2 = orc.make_params(cfg.U, cfg.V, cfg.Ws, cfg.Ht, cfg.height, cfg.block, cfg.window, 24, 48, geometry=wl.geometry(cfg), seed=cfg.seed, nthreads=1)
    data2, _, _ = orc.encode(lf, p2)
    assert data2 == data  # 1 thread vs all threads: byte-identical


def test_out_of_range_coordinates_decode_to_black_and_are_counted(enc):
    cfg, lf, data, info, s = enc("cfg1_lossy")
    coords = np.array([[0, 0, 0, 0], [8, 0, 0, 0], [0, -1, 0, 0], [0, 0, 64, 0], [0, 0, 0, 64], [7, 7, 63, 63]], dtype=np.int32)
    out, oob = s.decode(coords, return_oob=True)
    assert oob == 4 and not out[1:5].any()
    assert np.array_equal(out[0], info["p1"][0, 0, 0, 0]) and np.array_equal(out[5], info["p1"][7, 7, 63, 63])


def test_monotone_rate_and_quality():
    # raising tau never grows the stream; lowering tau never lowers PSNR (weakly)
    rng = np.random.default_rng(5)
    lf = random_lf(rng, 4, 4, 32, 32)
    p = orc.make_params(4, 4, 32, 32, 2, 4, 4)
    tree = orc.Tree(lf, p)
    sizes, q = [], []
    for tau in (0, 10, 30, 80, 200, 1000):
        tree.threshold(tau // 2, tau)
        sizes.append(len(tree.serialize()))
        q.append(orc.psnr(tree.reconstruct(), lf))
    assert all(a >= b for a, b in zip(sizes, sizes[1:]))
    assert all(a >= b - 1e-9 for a, b in zip(q, q[1:]))


def test_stats_locality_single_pixel(enc):
    # one pixel touches, per channel and level, its own block plus at most one
    # reference block through the MV: <= 2 h blocks per channel, independent of the stream size
    cfg, lf, data, info, s = enc("mini4")
    st = s.stats_decode(np.array([[5, 9, 17, 30]], dtype=np.int32))
    assert st["taps"] == 1 and st["rkv_bytes"] == 5
    assert st["blocks_touched"] <= 3 * 2 * cfg.height
    assert st["in_bytes"] == 16 and st["out_bytes"] == 3


def _bits15(N):
    """BISE bits per value in units of 1/15 bit, R15: the cheapest of plain 15 ceil(log2 N), trit 24 + 15 m, quint 35 + 15 m."""
    lay, m = PyStream.layout(N)
    return 15 * m if lay == 0 else (24 + 15 * m if lay == 1 else 35 + 15 * m)


@pytest.mark.parametrize("policy", [orc.POLICY_ADAPTIVE, orc.POLICY_ALL])
def test_stats_of_an_exhaustive_decode_equal_the_closed_form(policy):
    """SURVEY 8(d) D5 on a tau = 0 stream (every block significant) when EVERY pixel is decoded: each (plane-channel, block) is
    touched exactly once, so the counters have closed forms in terms of the directory, read here by the independent PyStream reader:
    flag bits = sum over plane-channels of nblk x (2 if predictive else 1); payload = sum of nblk x B^2 x bits/value(N); motion records
    = (number of predicted blocks) x bits/record; top-level RKV = U_h V_h Ws Ht x 5 bytes; plus 16 + 3 bytes per coordinate."""
    rng = np.random.default_rng(11)
    U, V, Ws, Ht, h, B, W = 3, 4, 16, 12, 2, 4, 3
    lf = random_lf(rng, U, V, Ws, Ht)
    data, info, tree = _encode(lf, h, B, W, 0, 0, policy)
    tree.close()
    ps, s = PyStream(data), orc.Stream(data)
    n = U * V * Ws * Ht
    cfg = wl.Config("x", U, V, Ws, Ht, h, 1, 0, 0, None, 0, Ws, Ht, 1, 0)
    st = s.stats_decode(wl.all_coords(cfg))
    flag_bits = pay15 = n_pred = 0
    for L in range(h):
        UL, VL = ps.dims[L]
        for pv in range(VL):
            for pu in range(UL):
                for c in range(3):
                    off, N, foff, poff, moff = ps.dirent(L, pu, pv, c)
                    isp = (pu | pv) & 1
                    assert all(ps.flag(foff, 0, b) for b in range(ps.nblk))          # tau = 0: every block stored
                    flag_bits += ps.nblk * (2 if isp else 1)
                    pay15 += ps.nblk * B * B * _bits15(N)
                    if isp:
                        n_pred += sum(ps.flag(foff, 1, b) for b in range(ps.nblk))
    nd = 2 * W + 1
    assert n_pred > 0 and (policy != orc.POLICY_ALL or n_pred == sum(ps.nblk * 3 for L in range(h) for pv in range(ps.dims[L][1])
                                                                     for pu in range(ps.dims[L][0]) if (pu | pv) & 1))
    assert st["blocks_touched"] == ps.n_pc * ps.nblk
    assert st["flag_bits"] == flag_bits
    assert st["payload_bits15"] == pay15
    assert st["mv_bits15"] == n_pred * _bits15(2 * nd * nd)
    assert st["rkv_bytes"] == ps.dims[h][0] * ps.dims[h][1] * Ws * Ht * 5
    assert (st["in_bytes"], st["out_bytes"], st["taps"]) == (16 * n, 3 * n, n)
    expect = (flag_bits + (pay15 + n_pred * _bits15(2 * nd * nd)) / 15.0) / 8.0 + st["rkv_bytes"] + 19 * n
    assert abs(st["bytes_alg"] - expect) < 1e-9 * expect


def test_stats_count_the_reference_block_reached_through_a_motion_vector():
    """One pixel whose block is predicted from a DIFFERENT block of the reference plane.  A gray 2 x 2 light field with Y planes
    128 + R, 128 + P, 128 - R, 128 - P has cluster mean 128, so its level-0 SRV images of Y are exactly R (reference) and P; P's
    block (0,0) is R's block (1,0) (P(x,y) = R(x+4,y)), which the search finds as subtractive (dx,dy) = (4,0), SAD 0.  Decoding pixel
    (u,v,s,t) = (1,0,1,2) must count, for Y, its own block (2 flag bits, 16 values, 1 motion record) and the reference block
    (1 flag bit, 16 values); for Co and Cg (all-zero SRVs: never predicted) the own block only."""
    rng = np.random.default_rng(3)
    R = rng.integers(-60, 61, (8, 8)).astype(np.int16)
    P = np.zeros((8, 8), dtype=np.int16)
    P[:, :4] = R[:, 4:]
    planes = [128 + R, 128 + P, 128 - R, 128 - P]
    lf = np.stack([np.repeat(p.astype(np.uint8)[..., None], 3, axis=-1) for p in planes]).reshape(2, 2, 8, 8, 3)
    data, info, tree = _encode(lf, 1, 4, 4, 0, 0, orc.POLICY_ADAPTIVE)
    assert tuple(tree.blocks(0, 1, 0, 0)[0, 0, :4]) == (0, 4, 0, 0)
    tree.close()
    ps, s = PyStream(data), orc.Stream(data)
    st = s.stats_decode(np.array([[1, 0, 1, 2]], dtype=np.int32))
    N_own = [ps.dirent(0, 1, 0, c)[1] for c in range(3)]
    N_ref = ps.dirent(0, 0, 0, 0)[1]
    assert st["blocks_touched"] == 4
    assert st["flag_bits"] == 2 + 1 + 2 + 2
    assert st["payload_bits15"] == 16 * (sum(_bits15(N) for N in N_own) + _bits15(N_ref))
    assert st["mv_bits15"] == _bits15(2 * 81) == 114          # N = 162: trit, m = 6: (8 + 30) bits / 5 records = 7.6 bits
    assert st["rkv_bytes"] == 5 and st["out_bytes"] == 3 and st["in_bytes"] == 16
    # the same pixel twice, and a second pixel of the same block: nothing new is counted (each distinct block once per batch)
    st2 = s.stats_decode(np.array([[1, 0, 1, 2], [1, 0, 1, 2], [1, 0, 2, 2]], dtype=np.int32))
    assert st2["blocks_touched"] == 4 and st2["payload_bits15"] == st["payload_bits15"] and st2["rkv_bytes"] == 10


def test_psnr_closed_form():
    # uniform error 1 -> 20 log10(255) = 48.1308 dB
    a = np.full((10, 10, 3), 100, dtype=np.uint8)
    assert abs(orc.psnr(a, a + 1) - 48.130803608679) < 1e-9
    assert orc.psnr(a, a) == float("inf")


# ---------------------------------------------------------------- progressive decoding (R26)
def _ycocg_planes_to_rgb(y, co, cg):
    t = y.astype(np.int32) - (cg.astype(np.int32) >> 1)
    g = cg + t
    b = t - (co.astype(np.int32) >> 1)
    r = b + co
    return np.clip(np.stack([r, g, b], axis=-1), 0, 255).astype(np.uint8)


def test_progressive_level_of_a_lossless_stream_is_the_cluster_key_view():
    """tau = 0: stopping the walk above level L yields exactly the representative key view X_L of the level-L cluster that
    contains the view (PAPER.md:200 defines X_L; the path-sum identity pins it) -- for every L in 0..h, every view."""
    import workloads as wl

    cfg = wl.CONFIGS["mini3"]                      # odd 5 x 5 grid, h = 3
    lf = wl.light_field(cfg)
    p = orc.make_params(cfg.U, cfg.V, cfg.Ws, cfg.Ht, cfg.height, cfg.block, cfg.window, 0, 0)
    data, info, tree = orc.encode(lf, p)
    s = orc.Stream(data)
    for L in range(cfg.height + 1):
        s.set_min_level(L)
        full = s.decode_full()
        for v in range(cfg.V):
            for u in range(cfg.U):
                X = [tree.plane("X", L, u >> L, v >> L, c) for c in range(3)]
                assert np.array_equal(full[v, u], _ycocg_planes_to_rgb(*X)), (L, u, v)
        if L == 0:
            assert np.array_equal(full, lf)
    with pytest.raises(orc.OracleError):
        s.set_min_level(cfg.height + 1)
    with pytest.raises(orc.OracleError):
        s.set_min_level(-1)
    tree.close()


def test_progressive_top_level_equals_huge_threshold_stream_and_quality_is_monotone(enc):
    cfg, lf, data, info, s0 = enc("mini2")
    s = orc.Stream(data)
    p = orc.make_params(cfg.U, cfg.V, cfg.Ws, cfg.Ht, cfg.height, cfg.block, cfg.window, 10 ** 6, 10 ** 6)
    data_top, _, tree = orc.encode(lf, p)           # every block insignificant: only the RKV chain survives
    tree.close()
    top_only = orc.Stream(data_top).decode_full()
    quality, touched = [], []
    import workloads as wl

    rc = wl.random_coords(cfg, 3000)
    for L in range(cfg.height + 1):
        s.set_min_level(L)
        full = s.decode_full()
        quality.append(orc.psnr(full, lf))
        touched.append(s.stats_decode(rc)["blocks_touched"])
        assert np.array_equal(s.decode(rc), full[rc[:, 1], rc[:, 0], rc[:, 3], rc[:, 2]])   # random access = dense, at every level
    assert np.array_equal(full, top_only)           # min_level = h
    assert all(a >= b for a, b in zip(quality, quality[1:])) and quality[0] > quality[-1] + 3.0
    assert all(a > b for a, b in zip(touched, touched[1:])) and touched[-1] == 0
