"""Host logic, no GPU: the packed slice-JDS streams (the HBM layout the AlgFAC kernel reads with bulk
async copies; csrc/amgdd_stream.hpp) decode back to the CSR they were
made from, way by way and block by block, for narrow and wide column indices, ragged rows, empty
rows, two row groups, an aux vector, and block sizes that force slices to be split across blocks."""
import numpy as np
import pytest

import paper_1906_10575_b200 as m

NO_ROW = 0xFFFF


def decode(stream, ways, block_bytes, wide, nrows, has_aux, n_real=None, window=256):
    """Decoder written from the layout comment of amgdd_stream.hpp (independent of the packer).
    Returns per-row lists of (column, value) in stored order and the aux vector; checks the way
    descriptors (block counts, the real-group prefix, the cut of the last block)."""
    raw = stream.tobytes()
    n_real = nrows if n_real is None else n_real
    rows = [[] for _ in range(nrows)]
    aux = np.full(nrows, np.nan)
    seen = np.zeros(nrows, dtype=int)
    cdt = np.uint32 if wide else np.uint16
    expect_off = 0
    load = []
    for w in range(len(ways)):
        wd = ways[w]
        nblocks, off = int(wd["nblocks"]), 16 * int(wd["off16"])
        assert off == expect_off, "ways are laid back to back"
        cur, real_slices, ghost_seen, last_real_block = None, 0, False, -1
        end = off
        for j in range(nblocks):
            base = off + j * block_bytes
            npieces, r0, r1, r2 = np.frombuffer(raw, dtype=np.uint32, count=4, offset=base)
            assert npieces >= 1 and r0 == 0 and r1 == 0 and r2 == 0
            end = base + 16 + 16 * int(npieces)
            for i in range(int(npieces)):
                poff, row_base = np.frombuffer(raw, dtype=np.uint32, count=2, offset=base + 16 + 16 * i)
                k0, nk, K, nnz = (int(t) for t in np.frombuffer(raw, dtype=np.uint16, count=4, offset=base + 16 + 16 * i + 8))
                assert poff % 16 == 0 and poff == end - base, "pieces are laid down back to back, 16-byte aligned"
                q = base + int(poff)
                if k0 == 0:
                    assert cur is None, "a new slice starts only after the previous one is complete"
                    rowid = np.frombuffer(raw, dtype=np.uint16, count=32, offset=q).astype(int)
                    lens = np.frombuffer(raw, dtype=np.uint16, count=32, offset=q + 64).astype(int)
                    q += 128
                    a = None
                    if has_aux:
                        a = np.frombuffer(raw, dtype=np.float64, count=32, offset=q)
                        q += 256
                    assert (np.diff(lens) <= 0).all(), "rows of a slice are sorted by descending length"
                    assert K == lens[0]
                    valid = rowid != NO_ROW
                    assert valid.any() and (lens[~valid] == 0).all() and valid[: valid.sum()].all(), "missing rows are the last lanes"
                    assert row_base % window == 0 or (row_base - n_real) % window == 0
                    grows = np.where(valid, int(row_base) + rowid, -1)
                    assert (rowid[valid] < window).all()
                    for jj in np.nonzero(valid)[0]:
                        assert seen[grows[jj]] == 0
                        seen[grows[jj]] = 1
                        if has_aux:
                            aux[grows[jj]] = a[jj]
                    is_real = bool((grows[valid] < n_real).all())
                    assert is_real or (grows[valid] >= n_real).all(), "the two groups never mix inside a slice"
                    assert not (is_real and ghost_seen), "inside a way the first group comes first"
                    ghost_seen = ghost_seen or not is_real
                    cur = dict(rows=grows, lens=lens, K=K, k=0, real=is_real)
                else:
                    assert i == 0 and cur is not None, "only piece 0 may continue a slice"
                    assert k0 == cur["k"] and K == cur["K"]
                vals = np.frombuffer(raw, dtype=np.float64, count=nnz, offset=q)
                cols = np.frombuffer(raw, dtype=cdt, count=nnz, offset=q + 8 * nnz)
                e = 0
                for k in range(k0, k0 + nk):
                    cnt = int((cur["lens"] > k).sum())
                    assert cnt >= 1
                    for jj in range(cnt):
                        rows[cur["rows"][jj]].append((int(cols[e + jj]), float(vals[e + jj])))
                    e += cnt
                assert e == nnz
                cur["k"] = k0 + nk
                end = q + ((nnz * (8 + cols.itemsize) + 15) // 16) * 16
                assert end - base <= block_bytes
                if cur["k"] == cur["K"]:
                    if cur["real"]:
                        real_slices += 1
                        last_real_block = j
                    cur = None
                else:
                    assert i == int(npieces) - 1, "a slice that continues must end its block"
            if j == nblocks - 1:
                assert end - base == 16 * int(wd["last16"]), "the last block of a way is cut at its padded end"
        assert cur is None
        assert int(wd["nslices_real"]) == real_slices and int(wd["nblocks_real"]) == last_real_block + 1
        expect_off = end
        load.append(end - off)
    assert expect_off == len(raw) and seen.all()
    return rows, aux, load


def random_csr(rng, nrows, ncols, max_len, empty_frac=0.1):
    lens = rng.integers(1, max_len + 1, size=nrows)
    lens[rng.random(nrows) < empty_frac] = 0
    rp = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    ci = np.concatenate([np.sort(rng.choice(ncols, size=k, replace=False)) for k in lens] + [np.zeros(0, int)]).astype(np.int32)
    v = rng.standard_normal(rp[-1])
    return rp, ci, v


def check_rows(rows, rp, ci, v):
    for i, r in enumerate(rows):
        cols = [c for c, _ in r]
        vals = [x for _, x in r]
        assert cols == ci[rp[i]:rp[i + 1]].tolist(), f"row {i}: columns (in stored order)"
        assert vals == v[rp[i]:rp[i + 1]].tolist(), f"row {i}: values"


@pytest.mark.parametrize("wide", [False, True])
@pytest.mark.parametrize("block_bytes", [1024, 2048, 8192])
def test_stream_round_trip(wide, block_bytes):
    rng = np.random.default_rng(7 + block_bytes + wide)
    ncols = 70000 if wide else 5000
    nrows, n_real = 3000, 2013
    rp, ci, v = random_csr(rng, nrows, ncols, 60)
    aux = rng.standard_normal(nrows)
    stream, ways = m.amgdd_pack_stream(rp, ci, v, wide=wide, block_bytes=block_bytes, n_real=n_real, aux=aux)
    assert len(ways) == m.NUM_WAYS and len(stream) % 16 == 0
    rows, aux2, load = decode(stream, ways, block_bytes, wide, nrows, True, n_real)
    check_rows(rows, rp, ci, v)
    assert np.array_equal(aux2, aux)
    # the ways are balanced: slices go to the lightest way, so no way exceeds the mean by more than a slice or so
    assert max(load) <= np.mean(load) + 32 * 60 * 12 + 1024
    # 10 (narrow) / 12 (wide) bytes per nonzero, nothing padded; per row 2 + 2 + 8 (rowid, len, aux);
    # per block a header, per piece a descriptor and padding to 16, and at most one step (<= 32
    # entries) that did not fit the tail of a block any more
    per_nnz = 12 if wide else 10
    ideal = rp[-1] * per_nnz
    nblocks = int(ways["nblocks"].sum())
    nslices = -(-n_real // 32) + -(-(nrows - n_real) // 32) + 30
    assert len(stream) <= ideal + nslices * (32 * 12 + 32) + nblocks * (16 + 2 * 32 + 32 * per_nnz)
    if block_bytes == 8192:
        assert len(stream) <= 1.08 * ideal


@pytest.mark.parametrize("window", [32, 64, 1024])
def test_windows_and_no_aux(window):
    rng = np.random.default_rng(window)
    rp, ci, v = random_csr(rng, 777, 3000, 25, empty_frac=0.3)
    stream, ways = m.amgdd_pack_stream(rp, ci, v, block_bytes=2048, window=window)
    rows, _, _ = decode(stream, ways, 2048, False, 777, False, window=window)
    check_rows(rows, rp, ci, v)
    assert np.array_equal(ways["nblocks"], ways["nblocks_real"])


def test_long_rows_are_split_across_blocks():
    # one row of 5000 entries (50 KB) in 1 KiB blocks, next to short rows
    rng = np.random.default_rng(3)
    lens = np.array([3, 5000, 0, 7, 2500] + [4] * 40)
    rp = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    ci = np.concatenate([np.sort(rng.choice(60000, size=k, replace=False)) for k in lens]).astype(np.int32)
    v = rng.standard_normal(rp[-1])
    stream, ways = m.amgdd_pack_stream(rp, ci, v, block_bytes=1024)
    assert ways["nblocks"].sum() > 50
    rows, _, _ = decode(stream, ways, 1024, False, len(lens), False)
    check_rows(rows, rp, ci, v)


def test_few_rows_and_empty_matrix():
    rp = np.array([0, 2, 2, 5], dtype=np.int32)
    ci = np.array([0, 3, 1, 2, 3], dtype=np.int32)
    v = np.arange(5, dtype=np.float64)
    stream, ways = m.amgdd_pack_stream(rp, ci, v)
    # one slice in way 0: block header + one descriptor + rowid/len + 5 entries padded to 16
    assert ways["nblocks"].tolist() == [1] + [0] * (m.NUM_WAYS - 1)
    assert len(stream) == 16 + 16 + 128 + ((5 * 10 + 15) // 16) * 16
    rows, _, _ = decode(stream, ways, 2048, False, 3, False)
    check_rows(rows, rp, ci, v)
    # a slice of empty rows still gets a piece (its rows still run their epilogue)
    stream, ways = m.amgdd_pack_stream(np.zeros(4, np.int32), np.zeros(0, np.int32), np.zeros(0))
    assert ways["nblocks"].sum() == 1 and len(stream) == 16 + 16 + 128
    rows, _, _ = decode(stream, ways, 2048, False, 3, False)
    assert rows == [[], [], []]
    stream, ways = m.amgdd_pack_stream(np.zeros(1, np.int32), np.zeros(0, np.int32), np.zeros(0))
    assert ways["nblocks"].sum() == 0 and len(stream) == 0


def test_bad_arguments():
    rp = np.array([0, 200], dtype=np.int32)
    ci = np.arange(200, dtype=np.int32)
    v = np.ones(200)
    with pytest.raises(m.AmgddError) as e:            # narrow form cannot hold column 70000
        m.amgdd_pack_stream(np.array([0, 1], np.int32), np.array([70000], np.int32), np.ones(1))
    assert e.value.code == -1
    with pytest.raises(m.AmgddError) as e:
        m.amgdd_pack_stream(rp, ci, v, block_bytes=1000)
    assert e.value.code == -1
    with pytest.raises(m.AmgddError) as e:
        m.amgdd_pack_stream(rp, ci, v, window=48)
    assert e.value.code == -1
    with pytest.raises(m.AmgddError) as e:
        m.amgdd_pack_stream(rp, ci, v, n_real=2)
    assert e.value.code == -1
    big = np.array([0, 70000], dtype=np.int32)        # more than 65535 entries in one row
    with pytest.raises(m.AmgddError) as e:
        m.amgdd_pack_stream(big, np.zeros(70000, np.int32), np.zeros(70000), wide=True)
    assert e.value.code == -9
