"""The oracle's hsma() was split into one routine per closure (round 2): the split must reproduce, bit for bit, what
the single-function body computed -- tests/golden/closure_results.txt was written by that body (its commit precedes
the split) through tests/golden/make_closure_golden.py, which calls only oracle/.  Also pins the deterministic
default wall / face points (reading S5b) directly.  `-m "not gpu"`."""
import importlib.util
import os

import numpy as np
import pytest

from oracle import hsma_oracle as O

HERE = os.path.dirname(os.path.abspath(__file__))


def _gen():
    spec = importlib.util.spec_from_file_location("make_closure_golden", os.path.join(HERE, "golden", "make_closure_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def _stored():
    out = {}
    with open(os.path.join(HERE, "golden", "closure_results.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            case, key, val = line.split()
            out.setdefault(case, {})[key] = float.fromhex(val)
    return out


GEN = _gen()
CASES = GEN.cases()


@pytest.mark.parametrize("name", sorted(CASES))
def test_split_oracle_is_bit_identical_to_the_single_function_body(name):
    w, kw = CASES[name]
    got = GEN.digest(O.hsma(w, **kw))
    want = _stored()[name]
    assert set(got) == set(want)
    for k in want:
        assert got[k] == want[k], (name, k, got[k], want[k])


def test_every_closure_routine_is_exercised():
    """One stored case at least per routine of the split."""
    seen = set()
    for w, _ in CASES.values():
        L = np.asarray(w.L, float)
        R0 = 0.5 * float(np.linalg.norm(L))
        cl = O.make_closure(w, L, R0, w.p)
        seen.add((w.kind, w.closure, cl.drop_constant, cl.far_cells is not None, cl.F.shape[0] > cl.check_targets.shape[0] // 2 + 1))
    assert len(seen) >= 7


# ---- default points on the faces (reading S5b): pinned by what the rule states, not by re-running it -------------------
@pytest.mark.parametrize("K,L,axes", [(1000, (1.0, 1.0, 1.0), (0, 1, 2)), (1500, (1.0, 1.0, 0.5), (0, 1, 2)), (600, (1.0, 1.0, 0.5), (2,)),
                                      (37, (1.0, 1.5, 0.7), (0, 1, 2))])
def test_default_face_points_lie_on_the_stated_faces_in_proportion_to_area_and_fill_them_evenly(K, L, axes):
    Lh = np.asarray(L)
    x = O.default_face_points(K, L, axes)
    assert x.shape == (K, 3)
    assert np.all(np.abs(x) <= 0.5 * Lh + 1e-15)
    on = np.isclose(np.abs(x), 0.5 * Lh, rtol=0, atol=1e-15)
    faces = [(a, s) for a in range(3) if a in axes for s in (-1, 1)]
    area = {(a, s): np.prod(np.delete(Lh, a)) for a, s in faces}
    tot = sum(area.values())
    counted = 0
    for (a, s) in faces:
        sel = on[:, a] & (np.sign(x[:, a]) == s)
        # a point of another face can touch this face's plane only on an edge: u or v would be exactly +-1/2 (never: frac != 0)
        n = int(sel.sum())
        counted += n
        assert abs(n - K * area[(a, s)] / tot) <= 1.0 + 1e-9            # floor + at most one leftover
        if n >= 30:                                                     # even filling: every cell of a 3 x 3 grid is hit,
            uv = np.delete(x[sel], a, axis=1) / np.delete(Lh, a) + 0.5  # and the star discrepancy stays low-discrepancy small
            h, _, _ = np.histogram2d(uv[:, 0], uv[:, 1], bins=3, range=[[0, 1], [0, 1]])
            assert h.min() >= 0.5 * n / 9 and h.max() <= 1.6 * n / 9
    assert counted == K
    assert len(np.unique(np.round(x, 12), axis=0)) == K                 # no repeated point


@pytest.mark.parametrize("K,L", [(500, (1.0, 1.0, 1.0)), (300, (1.0, 1.2, 0.9)), (10, (2.0, 2.0, 2.0))])
def test_default_lower_face_points_are_on_the_lower_faces_only(K, L):
    Lh = np.asarray(L)
    x = O.default_lower_face_points(K, L)
    assert x.shape == (K, 3)
    low = np.isclose(x, -0.5 * Lh, rtol=0, atol=1e-15)
    assert low.any(axis=1).all()                                        # each point on some face x_a = -L_a/2
    assert not np.isclose(x, 0.5 * Lh, rtol=0, atol=1e-12).any()        # none on an upper face (its partner goes there)
    area = np.array([np.prod(np.delete(Lh, a)) for a in range(3)])
    first_axis = np.argmax(low, axis=1)
    for a in range(3):
        assert abs(int((first_axis == a).sum()) - K * area[a] / area.sum()) <= 1.0 + 1e-9
    # the partners x + L_a e_a of the face-pair closure lie on the opposite faces
    xt = x.copy()
    xt[np.arange(K), first_axis] += Lh[first_axis]
    assert np.allclose(xt[np.arange(K), first_axis], 0.5 * Lh[first_axis], rtol=0, atol=1e-15)
