"""Host logic, no GPU: the packed SELL-32 group streams (the HBM layout the AlgFAC kernel reads with
coalesced 128-bit loads; csrc/amgdd_stream.hpp) decode back to the CSR
they were made from, way by way and slice by slice, for narrow and wide column indices, ragged
rows, empty rows, two row groups, row flags and several sort windows."""
import numpy as np
import pytest

import paper_1906_10575_b200 as m

NO_ROW = 0xFFFFFFFF


def header_bytes(wide):
    return m.HEADER_BYTES_WIDE if wide else m.HEADER_BYTES_NARROW


def decode(stream, ways, wide, nrows, n_real=None, window=256):
    """Decoder written from the layout comment of amgdd_stream.hpp (independent of the packer).
    Returns per-row lists of (column, value) in stored order and the bytes of each way; checks the
    way descriptors (offsets, the real-group prefix) and that padding is zero."""
    raw = stream.tobytes()
    n_real = nrows if n_real is None else n_real
    gb = m.GROUP_BYTES_WIDE if wide else m.GROUP_BYTES_NARROW
    HB = header_bytes(wide)
    rows = [None] * nrows
    flags = np.zeros(nrows, dtype=np.int64)
    decode.flags = flags
    load = []
    # groups of all ways come first, back to back; then the headers, each way 128-byte aligned
    off = 0
    for w in ways:
        assert 128 * int(w["grp_off128"]) == off
        off += int(w["ngroups"]) * gb
    for w in ways:
        assert 128 * int(w["hdr_off128"]) == off
        off = -(-(off + int(w["nslices"]) * HB) // 128) * 128
    assert off == len(raw)
    for w in ways:
        g = 128 * int(w["grp_off128"])
        h = 128 * int(w["hdr_off128"])
        groups_seen = real_groups = real_slices = 0
        ghost_seen = False
        for s in range(int(w["nslices"])):
            if wide:                   # 32 x { uint32 row, uint32 K | flag << 31 }
                hdr = np.frombuffer(raw, dtype=np.uint32, count=64, offset=h + s * HB).reshape(32, 2)
                rid, K, flag = hdr[:, 0].astype(np.int64), hdr[:, 1] & 0x7FFFFFFF, hdr[:, 1] >> 31
            else:                      # 32 x uint32  row | K << 16 | flag << 31, row 0xFFFF: none
                hdr = np.frombuffer(raw, dtype=np.uint32, count=32, offset=h + s * HB)
                rid = (hdr & 0xFFFF).astype(np.int64)
                rid[rid == 0xFFFF] = NO_ROW
                K, flag = (hdr >> 16) & 0x7FFF, hdr >> 31
            assert (K == K[0]).all() and K[0] >= 1, "every lane carries the slice's group count"
            K = int(K[0])
            valid = rid != NO_ROW
            assert valid.any() and valid[: valid.sum()].all(), "missing rows are the last lanes"
            assert (flag[~valid] == 0).all()
            is_real = bool((rid[valid] < n_real).all())
            assert is_real or (rid[valid] >= n_real).all(), "the two row groups never mix inside a slice"
            assert not (is_real and ghost_seen), "inside a way the first row group comes first"
            ghost_seen = ghost_seen or not is_real
            base = 0 if is_real else n_real
            assert len({(int(r) - base) // window for r in rid[valid]}) == 1, "a slice stays inside one sort window"
            vals = np.empty((32, 4 * K))
            cols = np.empty((32, 4 * K), dtype=np.int64)
            for kg in range(K):
                q = g + (groups_seen + kg) * gb
                vals[:, 4 * kg: 4 * kg + 2] = np.frombuffer(raw, dtype=np.float64, count=64, offset=q).reshape(32, 2)
                vals[:, 4 * kg + 2: 4 * kg + 4] = np.frombuffer(raw, dtype=np.float64, count=64, offset=q + 512).reshape(32, 2)
                cdt = np.uint32 if wide else np.uint16
                cols[:, 4 * kg: 4 * kg + 4] = np.frombuffer(raw, dtype=cdt, count=128, offset=q + 1024).reshape(32, 4)
            groups_seen += K
            if is_real:
                real_groups += K
                real_slices += 1
            for j in range(32):
                if not valid[j]:
                    assert (vals[j] == 0).all() and (cols[j] == 0).all()
                    continue
                r = int(rid[j])
                assert rows[r] is None, "every row is stored once"
                rows[r] = (cols[j], vals[j])
                flags[r] = flag[j]
        assert groups_seen == int(w["ngroups"]) and real_groups == int(w["ngroups_real"]) and real_slices == int(w["nslices_real"])
        load.append(int(w["ngroups"]) * gb + int(w["nslices"]) * HB)
    assert all(r is not None for r in rows)
    return rows, load


def random_csr(rng, nrows, ncols, max_len, empty_frac=0.1):
    lens = rng.integers(1, max_len + 1, size=nrows)
    lens[rng.random(nrows) < empty_frac] = 0
    rp = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    ci = np.concatenate([np.sort(rng.choice(ncols, size=k, replace=False)) for k in lens] + [np.zeros(0, int)]).astype(np.int32)
    v = rng.standard_normal(rp[-1])
    return rp, ci, v


def check_rows(rows, rp, ci, v):
    """Stored order = CSR order; everything past the end of a row is padding (0.0, column 0)."""
    for i, (cols, vals) in enumerate(rows):
        n = rp[i + 1] - rp[i]
        assert n <= len(cols), f"row {i} does not fit its slice"
        assert cols[:n].tolist() == ci[rp[i]:rp[i + 1]].tolist(), f"row {i}: columns (in stored order)"
        assert vals[:n].tolist() == v[rp[i]:rp[i + 1]].tolist(), f"row {i}: values"
        assert (cols[n:] == 0).all() and (vals[n:] == 0).all(), f"row {i}: padding"


@pytest.mark.parametrize("wide", [False, True])
def test_stream_round_trip(wide):
    rng = np.random.default_rng(7 + wide)
    ncols = 70000 if wide else 5000
    nrows, n_real = 3000, 2013
    rp, ci, v = random_csr(rng, nrows, ncols, 60)
    rf = (rng.random(nrows) < 0.4).astype(np.uint8)
    stream, ways = m.amgdd_pack_stream(rp, ci, v, wide=wide, n_real=n_real, row_flags=rf)
    assert len(ways) == m.NUM_WAYS and len(stream) % 128 == 0
    rows, load = decode(stream, ways, wide, nrows, n_real)
    check_rows(rows, rp, ci, v)
    assert np.array_equal(decode.flags, rf), "bit 31 of the header word carries the row's flag"
    HB = header_bytes(wide)
    # the ways are balanced: a slice goes to the lightest way, so no way exceeds the mean by more than one slice
    gb = m.GROUP_BYTES_WIDE if wide else m.GROUP_BYTES_NARROW
    assert max(load) <= np.mean(load) + 15 * gb + HB
    # rows are sorted by length inside windows of 256, so a slice is padded by less than the spread
    # of lengths over 32 consecutive sorted rows (60 / 8 here) plus the round-up to a group of 4
    per_nnz = 12 if wide else 10
    assert int(ways["ngroups"].sum()) * 128 <= rp[-1] + nrows * (60 / 8 + 3) + 2 * 32 * 60
    assert len(stream) <= 1.35 * rp[-1] * per_nnz + (nrows / 32 + 2) * HB + 16 * 128


def test_uniform_rows_are_not_padded():
    # the shape of the coarse composite levels: rows of nearly one length -> 10 bytes per nonzero + headers
    rng = np.random.default_rng(11)
    nrows = 4096
    lens = np.full(nrows, 36)
    rp = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    ci = np.concatenate([np.sort(rng.choice(6000, size=k, replace=False)) for k in lens]).astype(np.int32)
    v = rng.standard_normal(rp[-1])
    stream, ways = m.amgdd_pack_stream(rp, ci, v)
    assert int(ways["ngroups"].sum()) == nrows // 32 * 9
    assert len(stream) == nrows // 32 * (9 * m.GROUP_BYTES_NARROW + m.HEADER_BYTES_NARROW)
    rows, _ = decode(stream, ways, False, nrows)
    check_rows(rows, rp, ci, v)


@pytest.mark.parametrize("window", [32, 64, 1024])
def test_windows_and_no_aux(window):
    rng = np.random.default_rng(window)
    rp, ci, v = random_csr(rng, 777, 3000, 25, empty_frac=0.3)
    stream, ways = m.amgdd_pack_stream(rp, ci, v, window=window)
    rows, _ = decode(stream, ways, False, 777, window=window)
    check_rows(rows, rp, ci, v)
    assert (decode.flags == 0).all(), "streams packed without row flags carry none"
    assert np.array_equal(ways["ngroups"], ways["ngroups_real"]) and np.array_equal(ways["nslices"], ways["nslices_real"])


def test_long_rows():
    # one row of 5000 entries next to short rows: its slice has 1250 groups
    rng = np.random.default_rng(3)
    lens = np.array([3, 5000, 0, 7, 2500] + [4] * 40)
    rp = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    ci = np.concatenate([np.sort(rng.choice(60000, size=k, replace=False)) for k in lens]).astype(np.int32)
    v = rng.standard_normal(rp[-1])
    stream, ways = m.amgdd_pack_stream(rp, ci, v)
    assert int(ways["ngroups"].max()) == 1250
    rows, _ = decode(stream, ways, False, len(lens))
    check_rows(rows, rp, ci, v)


def test_few_rows_and_empty_matrix():
    rp = np.array([0, 2, 2, 5], dtype=np.int32)
    ci = np.array([0, 3, 1, 2, 3], dtype=np.int32)
    v = np.arange(5, dtype=np.float64)
    stream, ways = m.amgdd_pack_stream(rp, ci, v)
    # one slice in way 0: one group (longest row 3 <= 4 steps) and one header
    assert ways["ngroups"].tolist() == [1] + [0] * (m.NUM_WAYS - 1)
    assert len(stream) == m.GROUP_BYTES_NARROW + m.HEADER_BYTES_NARROW
    rows, _ = decode(stream, ways, False, 3)
    check_rows(rows, rp, ci, v)
    # a slice of empty rows still gets one (all padding) group: its rows still run their epilogue
    stream, ways = m.amgdd_pack_stream(np.zeros(4, np.int32), np.zeros(0, np.int32), np.zeros(0))
    assert ways["ngroups"].sum() == 1 and len(stream) == m.GROUP_BYTES_NARROW + m.HEADER_BYTES_NARROW
    rows, _ = decode(stream, ways, False, 3)
    assert all((c == 0).all() and (x == 0).all() for c, x in rows)
    stream, ways = m.amgdd_pack_stream(np.zeros(1, np.int32), np.zeros(0, np.int32), np.zeros(0))
    assert ways["ngroups"].sum() == 0 and len(stream) == 0


def test_bad_arguments():
    rp = np.array([0, 200], dtype=np.int32)
    ci = np.arange(200, dtype=np.int32)
    v = np.ones(200)
    with pytest.raises(m.AmgddError) as e:            # narrow form cannot hold column 70000
        m.amgdd_pack_stream(np.array([0, 1], np.int32), np.array([70000], np.int32), np.ones(1))
    assert e.value.code == -1
    with pytest.raises(m.AmgddError) as e:
        m.amgdd_pack_stream(rp, ci, v, window=48)
    assert e.value.code == -1
    with pytest.raises(m.AmgddError) as e:
        m.amgdd_pack_stream(rp, ci, v, n_real=2)
    assert e.value.code == -1
    with pytest.raises(m.AmgddError) as e:            # the narrow header holds a 16-bit row: 65536 rows need the wide form
        m.amgdd_pack_stream(np.zeros(65537, np.int32), np.zeros(0, np.int32), np.zeros(0))
    assert e.value.code == -1
    stream, ways = m.amgdd_pack_stream(np.zeros(65537, np.int32), np.zeros(0, np.int32), np.zeros(0), wide=True)
    assert int(ways["nslices"].sum()) == 2048 and len(stream) == 2048 * (m.GROUP_BYTES_WIDE + m.HEADER_BYTES_WIDE)
    big = np.array([0, 70000], dtype=np.int32)        # more than 65535 entries in one row
    with pytest.raises(m.AmgddError) as e:
        m.amgdd_pack_stream(big, np.zeros(70000, np.int32), np.zeros(70000), wide=True)
    assert e.value.code == -9
