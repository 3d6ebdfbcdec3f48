"""The library's universe / lattice expansion (include/mcdc.h mcdc_lattice_expand*, DESIGN.md Appendix K) without a GPU:
it is host code, so its output can be held byte for byte to the hand-written config 3 and to the oracle's own,
independently written expansion (oracle/lattice.py)."""
import copy

import numpy as np
import pytest

from workloads import configs as W

KEYS = ("surf_coef", "surf_bc", "cell_offset", "hs_surface", "hs_sense", "cell_material")


@pytest.fixture(scope="module")
def M():
    from paper_2409_04668_b200 import build as b
    b.build()
    import paper_2409_04668_b200 as M
    return M


def test_config3_as_a_lattice_gives_the_hand_written_tables_byte_for_byte(M):
    hand = W.config3_pin_lattice()
    lat = W.config3_lattice().meta["lattice"]
    assert M.mcdc_lattice_expand_size(lat) == (hand.n_surfaces, hand.n_cells, len(hand.hs_surface)) == (327, 578, 2890)
    e = M.mcdc_lattice_expand(lat)
    for k in KEYS:
        a, b = np.ascontiguousarray(getattr(hand, k)), e[k]
        assert a.shape == b.shape and a.tobytes() == b.astype(a.dtype).tobytes(), k


def test_library_and_oracle_expansions_agree_on_the_mixed_lattice(M):
    from oracle import expand_lattice
    lat = W.lattice_mixed().meta["lattice"]
    e, o = M.mcdc_lattice_expand(lat), expand_lattice(lat)
    for k in KEYS:
        assert e[k].shape == o[k].shape and e[k].tobytes() == o[k].astype(e[k].dtype).tobytes(), k


def test_malformed_lattices_are_refused_by_the_library(M):
    base = W.lattice_mixed().meta["lattice"]
    for edit in (lambda l: l.__setitem__("fill", [[0, 1, 2, 3], [2, 0, 0, 1], [0, 2, 1, 0]]),
                 lambda l: l.__setitem__("fill", [[0, 1, 2, 0], [2, 0, 0, 1]]),
                 lambda l: l.__setitem__("pitch_y", -1.0),
                 lambda l: l.__setitem__("z_hi", l["z_lo"]),
                 lambda l: l.__setitem__("bc", [0, 1, 2, 3, 0, 0]),
                 lambda l: l["universes"][1]["cells"].__setitem__(0, ([(0, +1)], 2)),
                 lambda l: l["universes"][1]["cells"].__setitem__(0, ([(-7, +1)], 2)),
                 lambda l: l["universes"][1]["cells"].__setitem__(0, ([(-1, 0)], 2)),
                 lambda l: l["universes"][1]["cells"].__setitem__(0, ([], 2))):
        lat = copy.deepcopy(base)
        edit(lat)
        with pytest.raises(M.McdcError) as ex:
            M.mcdc_lattice_expand(lat)
        assert ex.value.code == -3


def test_a_lattice_whose_element_count_overflows_int32_is_refused_by_all_three_calls(M):
    """nx * ny = 46341^2 > INT32_MAX used to wrap negative in int arithmetic: the fill check was skipped and the expansion
    went on to size its tables from garbage.  All three entry points now share one 64-bit guard."""
    import ctypes as C
    from paper_2409_04668_b200 import api
    lat = W.lattice_mixed().meta["lattice"]
    d, keep = api._make_lattice(lat)
    d.nx = d.ny = 46341                                   # fill is NOT that large: the guard must fire before it is read
    n = [C.c_int32() for _ in range(3)]
    assert M.lib().mcdc_lattice_expand_size(C.byref(d), *[C.byref(v) for v in n]) == -3
    buf_d, buf_i = (C.c_double * 16)(), (C.c_int32 * 16)()
    assert M.lib().mcdc_lattice_expand(C.byref(d), buf_d, buf_i, buf_i, buf_i, buf_i, buf_i) == -3
    pd, keep2 = api._make_desc(W.lattice_mixed())
    h = C.c_void_p()
    assert M.lib().mcdc_problem_create_lattice(C.byref(pd), C.byref(d), C.byref(h)) == -3 and not h.value
