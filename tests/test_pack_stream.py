"""Host logic, no GPU: the packed slice-JDS stream (the HBM layout the AlgFAC kernel reads with bulk
async copies; csrc/amgdd_stream.hpp) decodes back to the CSR it was
made from, chunk by chunk, for narrow and wide column indices, ragged rows, empty rows, two row
groups, an aux vector, and chunk sizes that force slices to be split across many chunks."""
import numpy as np
import pytest

import paper_1906_10575_b200 as m

NO_ROW = 0xFFFF


def decode(stream, nchunks, chunk_bytes, wide, nrows, has_aux, n_real=None, window=256):
    """Decoder written from the layout comment of amgdd_stream.hpp (independent of the packer).
    Returns per-row lists of (column, value) in stored order, the aux vector, and the chunk index
    in which the last slice of the first group ends."""
    raw = stream.tobytes()
    n_real = nrows if n_real is None else n_real
    rows = [[] for _ in range(nrows)]
    aux = np.full(nrows, np.nan)
    seen = np.zeros(nrows, dtype=int)
    cdt = np.uint32 if wide else np.uint16
    next_slice, cur, last_real_chunk = 0, None, -1          # cur: state of the slice being read
    for c in range(nchunks):
        base = c * chunk_bytes
        npieces, slice0, r0, r1 = np.frombuffer(raw, dtype=np.uint32, count=4, offset=base)
        assert npieces >= 1 and r0 == 0 and r1 == 0
        end = base + 16 + 16 * int(npieces)
        for i in range(int(npieces)):
            off, row_base = np.frombuffer(raw, dtype=np.uint32, count=2, offset=base + 16 + 16 * i)
            k0, nk, K, nnz = (int(t) for t in np.frombuffer(raw, dtype=np.uint16, count=4, offset=base + 16 + 16 * i + 8))
            assert off % 16 == 0 and off == end - base, "pieces are laid down back to back, 16-byte aligned"
            q = base + int(off)
            if k0 == 0:
                assert cur is None, "a new slice starts only after the previous one is complete"
                assert int(slice0) + i == next_slice
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
                assert (lens[~valid] == 0).all() and valid[: valid.sum()].all(), "missing rows are the last lanes"
                assert row_base % window == 0 or row_base == n_real or (row_base - n_real) % window == 0
                grows = np.where(valid, int(row_base) + rowid, -1)
                assert (rowid[valid] < window).all()
                for j in np.nonzero(valid)[0]:
                    assert seen[grows[j]] == 0
                    seen[grows[j]] = 1
                    if has_aux:
                        aux[grows[j]] = a[j]
                # both groups never mix inside a slice
                assert (grows[valid] < n_real).all() or (grows[valid] >= n_real).all()
                cur = dict(rows=grows, lens=lens, K=K, k=0, real=bool((grows[valid] < n_real).all()) if valid.any() else False)
                next_slice += 1
            else:
                assert i == 0 and cur is not None and int(slice0) == next_slice - 1, "only piece 0 may continue a slice"
                assert k0 == cur["k"] and K == cur["K"]
            vals = np.frombuffer(raw, dtype=np.float64, count=nnz, offset=q)
            cols = np.frombuffer(raw, dtype=cdt, count=nnz, offset=q + 8 * nnz)
            e = 0
            for k in range(k0, k0 + nk):
                cnt = int((cur["lens"] > k).sum())
                assert cnt >= 1
                for j in range(cnt):
                    rows[cur["rows"][j]].append((int(cols[e + j]), float(vals[e + j])))
                e += cnt
            assert e == nnz
            cur["k"] = k0 + nk
            end = q + ((nnz * (8 + cols.itemsize) + 15) // 16) * 16
            assert end - base <= chunk_bytes
            if cur["k"] == cur["K"]:
                if cur["real"]:
                    last_real_chunk = c
                cur = None
            else:
                assert i == int(npieces) - 1, "a slice that continues must end its chunk"
        if c == nchunks - 1:
            assert len(raw) == end                                   # the last chunk is cut at its padded end
    assert cur is None and seen.all()
    return rows, aux, last_real_chunk


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
@pytest.mark.parametrize("chunk_bytes", [1024, 4096, 16384])
def test_stream_round_trip(wide, chunk_bytes):
    rng = np.random.default_rng(7 + chunk_bytes + wide)
    ncols = 70000 if wide else 5000
    nrows, n_real = 1500, 1013
    rp, ci, v = random_csr(rng, nrows, ncols, 60)
    aux = rng.standard_normal(nrows)
    stream, nchunks, nreal = m.amgdd_pack_stream(rp, ci, v, wide=wide, chunk_bytes=chunk_bytes, n_real=n_real, aux=aux)
    assert nchunks >= 2 and len(stream) % 16 == 0
    rows, aux2, last_real = decode(stream, nchunks, chunk_bytes, wide, nrows, True, n_real)
    check_rows(rows, rp, ci, v)
    assert np.array_equal(aux2, aux)
    assert nreal == last_real + 1
    # 10 (narrow) / 12 (wide) bytes per nonzero, nothing padded; per row 2 + 2 + 8 (rowid, len, aux);
    # per chunk a header, and per piece a descriptor and padding to 16
    per_nnz = 12 if wide else 10
    nslices = -(-n_real // 32) + -(-(nrows - n_real) // 32) + 10
    ideal = rp[-1] * per_nnz
    assert len(stream) <= ideal + nslices * (32 * 12 + 32) + nchunks * (16 + 2 * 32 + per_nnz * 32)
    if chunk_bytes == 16384:
        assert len(stream) <= 1.08 * ideal


@pytest.mark.parametrize("window", [32, 64, 1024])
def test_windows_and_no_aux(window):
    rng = np.random.default_rng(window)
    rp, ci, v = random_csr(rng, 777, 3000, 25, empty_frac=0.3)
    stream, nchunks, nreal = m.amgdd_pack_stream(rp, ci, v, chunk_bytes=2048, window=window)
    rows, _, last_real = decode(stream, nchunks, 2048, False, 777, False, window=window)
    check_rows(rows, rp, ci, v)
    assert nreal == nchunks == last_real + 1


def test_long_rows_are_split_across_chunks():
    # one row of 5000 entries (50 KB) in 1 KiB chunks, next to short rows
    rng = np.random.default_rng(3)
    lens = np.array([3, 5000, 0, 7, 2500] + [4] * 40)
    rp = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    ci = np.concatenate([np.sort(rng.choice(60000, size=k, replace=False)) for k in lens]).astype(np.int32)
    v = rng.standard_normal(rp[-1])
    stream, nchunks, _ = m.amgdd_pack_stream(rp, ci, v, chunk_bytes=1024)
    assert nchunks > 50
    rows, _, _ = decode(stream, nchunks, 1024, False, len(lens), False)
    check_rows(rows, rp, ci, v)


def test_single_chunk_and_empty_matrix():
    rp = np.array([0, 2, 2, 5], dtype=np.int32)
    ci = np.array([0, 3, 1, 2, 3], dtype=np.int32)
    v = np.arange(5, dtype=np.float64)
    stream, nchunks, nreal = m.amgdd_pack_stream(rp, ci, v)
    # header + one descriptor + rowid/len + 5 entries padded to 16
    assert nchunks == 1 and nreal == 1 and len(stream) == 16 + 16 + 128 + ((5 * 10 + 15) // 16) * 16
    rows, _, _ = decode(stream, nchunks, 16384, False, 3, False)
    check_rows(rows, rp, ci, v)
    # a slice of empty rows still gets a piece (its rows still run their epilogue)
    stream, nchunks, _ = m.amgdd_pack_stream(np.zeros(4, np.int32), np.zeros(0, np.int32), np.zeros(0))
    assert nchunks == 1 and len(stream) == 16 + 16 + 128
    rows, _, _ = decode(stream, nchunks, 16384, False, 3, False)
    assert rows == [[], [], []]
    stream, nchunks, _ = m.amgdd_pack_stream(np.zeros(1, np.int32), np.zeros(0, np.int32), np.zeros(0))
    assert nchunks == 0 and len(stream) == 0


def test_bad_arguments():
    rp = np.array([0, 200], dtype=np.int32)
    ci = np.arange(200, dtype=np.int32)
    v = np.ones(200)
    with pytest.raises(m.AmgddError) as e:            # narrow form cannot hold column 70000
        m.amgdd_pack_stream(np.array([0, 1], np.int32), np.array([70000], np.int32), np.ones(1))
    assert e.value.code == -1
    with pytest.raises(m.AmgddError) as e:
        m.amgdd_pack_stream(rp, ci, v, chunk_bytes=1000)
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
