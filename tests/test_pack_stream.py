"""Host logic, no GPU: the packed CSR stream (the HBM layout the AlgFAC kernel reads with bulk
async copies; csrc/amgdd_stream.hpp) decodes back to the CSR it was
made from, chunk by chunk, for narrow and wide column indices, ragged rows, empty rows and
chunk sizes that force many chunk boundaries."""
import numpy as np
import pytest

import paper_1906_10575_b200 as m


def decode(stream, nchunks, chunk_bytes, wide):
    """Decoder written from the layout comment of amgdd_stream.hpp (independent of the packer)."""
    rows_seen, rp, ci, v = 0, [0], [], []
    raw = stream.tobytes()
    for c in range(nchunks):
        base = c * chunk_bytes
        row_begin, nrows, nnz, reserved = np.frombuffer(raw, dtype=np.int32, count=4, offset=base)
        assert reserved == 0 and row_begin == rows_seen and nrows >= 1
        vals = np.frombuffer(raw, dtype=np.float64, count=nnz, offset=base + 16)
        cdt = np.uint32 if wide else np.uint16
        cols = np.frombuffer(raw, dtype=cdt, count=nnz, offset=base + 16 + 8 * nnz)
        rowend = np.frombuffer(raw, dtype=np.uint16, count=nrows, offset=base + 16 + 8 * nnz + cols.itemsize * nnz)
        used = 16 + 8 * nnz + cols.itemsize * nnz + 2 * nrows
        assert used <= chunk_bytes
        assert (np.diff(np.concatenate([[0], rowend.astype(np.int64)])) >= 0).all()
        assert rowend[-1] == nnz
        start = rp[-1]                                              # row pointers from the chunk-local ends
        rp.extend((start + rowend.astype(np.int64)).tolist())
        ci.extend(cols.astype(np.int64).tolist())
        v.extend(vals.tolist())
        rows_seen += nrows
        if c == nchunks - 1:
            assert len(raw) == base + ((used + 15) // 16) * 16      # the last chunk is cut at its padded end
    return np.array(rp), np.array(ci), np.array(v)


def random_csr(rng, nrows, ncols, max_len, empty_frac=0.1):
    lens = rng.integers(1, max_len + 1, size=nrows)
    lens[rng.random(nrows) < empty_frac] = 0
    rp = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    ci = np.concatenate([np.sort(rng.choice(ncols, size=k, replace=False)) for k in lens] + [np.zeros(0, int)]).astype(np.int32)
    v = rng.standard_normal(rp[-1])
    return rp, ci, v


@pytest.mark.parametrize("wide", [False, True])
@pytest.mark.parametrize("chunk_bytes", [1024, 4096, 16384])
def test_stream_round_trip(wide, chunk_bytes):
    rng = np.random.default_rng(7 + chunk_bytes + wide)
    ncols = 70000 if wide else 5000
    rp, ci, v = random_csr(rng, 1500, ncols, 60)
    stream, nchunks = m.amgdd_pack_stream(rp, ci, v, wide=wide, chunk_bytes=chunk_bytes)
    assert nchunks >= 2 and len(stream) % 16 == 0
    rp2, ci2, v2 = decode(stream, nchunks, chunk_bytes, wide)
    assert np.array_equal(rp2, rp) and np.array_equal(ci2, ci) and np.array_equal(v2, v)
    # 10 (narrow) / 12 (wide) bytes per nonzero + 2 per row; per chunk a 16-byte header, padding
    # to 16 and at most one row that did not fit any more (greedy packing)
    per_nnz = 12 if wide else 10
    ideal = rp[-1] * per_nnz + 2 * (len(rp) - 1)
    assert len(stream) <= ideal + nchunks * (16 + 16 + 60 * per_nnz + 2)
    if chunk_bytes == 16384:
        assert len(stream) <= 1.03 * ideal


def test_single_chunk_and_empty_matrix():
    rp = np.array([0, 2, 2, 5], dtype=np.int32)
    ci = np.array([0, 3, 1, 2, 3], dtype=np.int32)
    v = np.arange(5, dtype=np.float64)
    stream, nchunks = m.amgdd_pack_stream(rp, ci, v)
    assert nchunks == 1 and len(stream) == ((16 + 5 * 10 + 3 * 2 + 15) // 16) * 16
    rp2, ci2, v2 = decode(stream, nchunks, 16384, False)
    assert np.array_equal(rp2, rp) and np.array_equal(ci2, ci) and np.array_equal(v2, v)
    stream, nchunks = m.amgdd_pack_stream(np.zeros(1, np.int32), np.zeros(0, np.int32), np.zeros(0))
    assert nchunks == 0 and len(stream) == 0


def test_row_too_long_and_bad_arguments():
    n = 200                                           # 16 + 200*10 + 2 > 1024
    rp = np.array([0, n], dtype=np.int32)
    ci = np.arange(n, dtype=np.int32)
    v = np.ones(n)
    with pytest.raises(m.AmgddError) as e:
        m.amgdd_pack_stream(rp, ci, v, chunk_bytes=1024)
    assert e.value.code == -9
    stream, nchunks = m.amgdd_pack_stream(rp, ci, v, chunk_bytes=4096)
    assert nchunks == 1
    with pytest.raises(m.AmgddError) as e:            # narrow form cannot hold column 70000
        m.amgdd_pack_stream(np.array([0, 1], np.int32), np.array([70000], np.int32), np.ones(1))
    assert e.value.code == -1
    with pytest.raises(m.AmgddError) as e:
        m.amgdd_pack_stream(rp, ci, v, chunk_bytes=1000)
    assert e.value.code == -1
