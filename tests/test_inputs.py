"""The torch transcription of the R-MAT recipe (paper_2606_01693_b200/inputs.py) produces the arrays of the numpy one."""
import numpy as np
import pytest

from paper_2606_01693_b200 import inputs

torch = pytest.importorskip("torch")


@pytest.mark.parametrize("scale,seed", [(6, 1), (10, 3), (12, 12)])
def test_rmat_torch_equals_numpy(scale, seed):
    rowptr, col, src = inputs.rmat_csr(scale, 16, seed=seed)
    t_rowptr, t_col, t_src = inputs.rmat_csr_torch(scale, 16, seed=seed, device="cpu", chunk=1 << 13)
    assert src == t_src
    assert np.array_equal(rowptr.astype(np.int64), t_rowptr.numpy())
    assert np.array_equal(col, t_col.numpy().view(np.uint32))


def test_rmat_shape_properties():
    rowptr, col, src = inputs.rmat_csr(10, 16, seed=1)
    nv = 1 << 10
    assert len(rowptr) == nv + 1 and rowptr[0] == 0 and rowptr[-1] == len(col)
    rows = np.repeat(np.arange(nv), np.diff(rowptr.astype(np.int64)))
    assert (rows != col).all()                                                  # no self-loops
    keys = rows.astype(np.int64) << 32 | col.astype(np.int64)
    assert (np.diff(keys) > 0).all()                                            # sorted, deduplicated
    assert set(zip(rows.tolist(), col.tolist())) == set(zip(col.tolist(), rows.tolist()))   # symmetric
    assert rowptr[src + 1] > rowptr[src]
