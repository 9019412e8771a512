"""CPU-side checks of the boundary: libgm.so builds/loads without a GPU, exports every symbol that
include/gm.h declares, and its host-only logic (workspace sizing, argument validation, the SFC cell
order) behaves as the header says.  No compute call is made here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def gm():
    from paper_1310_2041_b200 import build
    build.build()
    from paper_1310_2041_b200 import gm as g
    g.lib()
    return g


def header_functions():
    src = open(os.path.join(ROOT, "include", "gm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gm_[a-z_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(gm):
    names = header_functions()
    assert len(names) >= 16 and "gm_step" in names and "gm_energies" in names
    L = gm.lib()
    for n in names:
        assert hasattr(L, n), f"libgm.so does not export {n}"
    assert sorted(gm.SYMBOLS) == names          # the binding covers the same set, same names


def test_no_torch_types_in_the_abi():
    src = open(os.path.join(ROOT, "include", "gm.h")).read()
    assert "torch" not in re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    assert "at::" not in src and "Tensor" not in src


def base_cfg(gm, n=1000, box=12.0):
    c = gm.gm_config()
    c.struct_size = C.sizeof(gm.gm_config)
    c.n_particles = n
    c.n_types = 1
    c.max_bonds_per_particle = 2
    c.box[0] = c.box[1] = c.box[2] = box
    c.r_cut_max, c.r_skin, c.dt = 1.12, 0.4, 0.005
    c.pair_style, c.bond_style, c.integrator = 1, 1, 0
    return c


def test_query_workspace_scales_with_n_and_rejects_bad_configs(gm):
    small = gm.gm_query_workspace(base_cfg(gm, 1000))
    big = gm.gm_query_workspace(base_cfg(gm, 8000, 24.0))
    assert 0 < small < big
    assert big > 8000 * (16 * 8)                # at least the float4 arrays
    c = base_cfg(gm); c.struct_size = 12
    with pytest.raises(gm.GmError) as e:
        gm.gm_query_workspace(c)
    assert e.value.status == gm.GM_ERR_INVALID_ARG
    c = base_cfg(gm); c.n_types = 99
    with pytest.raises(gm.GmError):
        gm.gm_query_workspace(c)
    c = base_cfg(gm, box=4.0)                   # 4.0 < 3 * (1.12 + 0.4): the 27-cell search needs 3 cells
    with pytest.raises(gm.GmError) as e:
        gm.gm_query_workspace(c)
    assert e.value.status == gm.GM_ERR_BOX_TOO_SMALL
    c = base_cfg(gm); c.dt = 0.0
    with pytest.raises(gm.GmError):
        gm.gm_query_workspace(c)


def test_create_rejects_null_workspace_without_touching_cuda(gm):
    c = base_cfg(gm)
    h = C.c_void_p(0)
    st = gm.lib().gm_create(C.byref(c), None, 1 << 30, C.byref(h))
    assert st == gm.GM_ERR_INVALID_ARG and not h.value
    assert gm.lib().gm_last_error(None) is not None


def test_sfc_cell_order_is_a_hilbert_permutation(gm):
    # a permutation of the cells for any grid; cells run along x inside a row, and on a 2^k grid
    # consecutive (y, z) rows are edge neighbors (2-D Hilbert curve over the rows)
    for nc in ([8, 8, 8], [5, 7, 3], [13, 13, 13]):
        r = gm.gm_sfc_cell_order(nc)
        assert sorted(r.tolist()) == list(range(nc[0] * nc[1] * nc[2]))
        r3 = r.reshape(nc[2], nc[1], nc[0]).astype(np.int64)
        assert (np.diff(r3, axis=2) == 1).all()            # x-adjacent cells are memory neighbors
        assert (r3[:, :, 0] % nc[0] == 0).all()
    r = gm.gm_sfc_cell_order([4, 8, 8]).reshape(8, 8, 4)
    row = (r[:, :, 0] // 4).astype(np.int64)            # rank of row (z, y)
    inv = np.argsort(row.reshape(-1))
    zy = np.stack([inv // 8, inv % 8], axis=1)
    assert (np.abs(np.diff(zy, axis=0)).sum(axis=1) == 1).all()
    # locality on a clipped grid: the mean jump between consecutive rows stays close to 1 row
    r = gm.gm_sfc_cell_order([3, 13, 13]).reshape(13, 13, 3)
    inv = np.argsort((r[:, :, 0] // 3).reshape(-1))
    zy = np.stack([inv // 13, inv % 13], axis=1)
    assert np.abs(np.diff(zy, axis=0)).sum(axis=1).mean() < 1.5
