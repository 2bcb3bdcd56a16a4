"""Pins of the paper-exact Level-1 indexer oracle (oracle/l1_oracle.py; Eq.(1)-(5), (13)):
a hand-computed case, closed forms, a brute-force restatement of the selection rule, and invariants."""
import json
import os

import numpy as np
import pytest

from oracle.l1_oracle import (l1_chunk_scores, l1_entry_scores, l1_index_select, l1_query, l1_select, sigmoid,
                              validate_l1_selection)

HERE = os.path.dirname(os.path.abspath(__file__))


def test_hand_case():
    g = json.load(open(os.path.join(HERE, "golden", "l1_hand_case.json")))
    a = lambda k: np.array(g[k], dtype=np.float32)
    q, w = l1_query(a("h"), a("W_dq"), a("W_iuq"), a("W_w"), g["n_h"])
    np.testing.assert_allclose(q, g["q"], atol=1e-15)
    np.testing.assert_allclose(w, g["w"], atol=1e-15)
    I, pre = l1_entry_scores(q, w, a("index_k"))
    np.testing.assert_allclose(pre, g["pre"], atol=1e-15)
    np.testing.assert_allclose(I, g["I"], atol=1e-12)
    sel, _ = l1_select(l1_chunk_scores([I], 1), 4)
    assert sel.tolist() == g["select_C1_k4"]                     # pre == 0 -> I == 0.5 IS recalled (Eq.5 ">=")
    cs = l1_chunk_scores([I], 2)
    np.testing.assert_allclose(cs, g["chunk_score_C2"], atol=1e-12)
    assert l1_select(cs, 1)[0].tolist() == g["select_C2_k1"]


def test_closed_forms():
    g = np.random.default_rng(3)
    d, d_c, c_I, n_h, n = 12, 6, 4, 3, 50
    h = g.standard_normal(d).astype(np.float32)
    W_dq = g.standard_normal((d_c, d)).astype(np.float32)
    W_iuq = g.standard_normal((n_h * c_I, d_c)).astype(np.float32)
    W_w = g.standard_normal((n_h, d)).astype(np.float32)
    K = g.standard_normal((n, c_I)).astype(np.float32)
    q, w = l1_query(h, W_dq, W_iuq, W_w, n_h)
    # Eq.(1)-(2) compose to one linear map; Eq.(3) is a plain matvec (paper's row-vector form h . W)
    np.testing.assert_allclose(q.reshape(-1), h.astype(np.float64) @ (W_dq.astype(np.float64).T @ W_iuq.astype(np.float64).T), rtol=1e-12)
    np.testing.assert_allclose(w, h.astype(np.float64) @ W_w.astype(np.float64).T, rtol=1e-12)
    I, pre = l1_entry_scores(q, w, K)
    # element-wise restatement of Eq.(4) with python loops
    for s in range(0, n, 7):
        acc = 0.0
        for hh in range(n_h):
            acc += w[hh] * max(0.0, float(np.dot(q[hh], K[s].astype(np.float64))))
        assert pre[s] == pytest.approx(acc, rel=1e-12, abs=1e-12)
        assert I[s] == pytest.approx(1.0 / (1.0 + np.exp(-acc)), rel=1e-12)
    # one head, unit weight, positive match: I = sigmoid(q . k); negative match: ReLU gates it to I = 0.5
    q1, w1 = np.array([[1.0, 2.0]]), np.array([1.0])
    I1, _ = l1_entry_scores(q1, w1, np.array([[3.0, 1.0], [-3.0, -1.0]], dtype=np.float32))
    assert I1[0] == pytest.approx(1 / (1 + np.exp(-5.0))) and I1[1] == 0.5
    # all head weights zero: every entry scores exactly 0.5 and is recalled (threshold is ">=")
    I0, _ = l1_entry_scores(q, np.zeros(n_h), K)
    assert np.all(I0 == 0.5) and l1_select(l1_chunk_scores([I0], 8), 100)[0].tolist()[:7] == list(range(7))
    # sigmoid is monotone: I >= 0.5  <=>  pre >= 0; scaling w by a positive factor keeps the recalled set
    assert np.array_equal(I >= 0.5, pre >= 0)
    I2, _ = l1_entry_scores(q, 3.0 * w, K)
    assert np.array_equal(I >= 0.5, I2 >= 0.5)


def test_selection_rule_brute_force():
    g = np.random.default_rng(5)
    for trial in range(40):
        n, C, L = int(g.integers(1, 60)), int(g.integers(1, 9)), int(g.integers(1, 4))
        Is = [sigmoid(g.standard_normal(n) * 2 - 0.5) for _ in range(L)]
        if trial % 5 == 0:
            Is[0][: n // 2] = Is[0][0]                                 # ties
        cs = l1_chunk_scores(Is, C)
        n_chunks = (n + C - 1) // C
        # Eq.(13): union over layers of Eq.(5) sets, entry level, then "recall is in pages"
        entries = set()
        for I in Is:
            entries |= {s for s in range(n) if I[s] >= 0.5}
        chunks = sorted({s // C for s in entries})
        assert chunks == [c for c in range(n_chunks) if cs[c] >= 0.5]
        for k in (1, 3, n_chunks + 2):
            sel, val = l1_select(cs, k)
            want = sorted(chunks, key=lambda c: (-cs[c], c))[:k]
            assert [c for c in sel.tolist() if c >= 0] == want
            assert np.all(val[: len(want)] == cs[want]) and np.all(sel[len(want):] == -1)
            assert validate_l1_selection(sel, cs, k, 0.5, 1e-9) is None


def test_full_path_planted():
    """Planted structure: entries aligned with a positively-weighted head's query score high, the rest low."""
    g = np.random.default_rng(7)
    d, d_c, c_I, n_h, C, n = 32, 16, 8, 4, 4, 64
    h = g.standard_normal(d).astype(np.float32)
    layers, Ks, planted = [], [], set()
    for l in range(2):
        W_dq = (g.standard_normal((d_c, d)) / np.sqrt(d)).astype(np.float32)
        W_iuq = (g.standard_normal((n_h * c_I, d_c)) / np.sqrt(d_c)).astype(np.float32)
        W_w = np.zeros((n_h, d), dtype=np.float32)
        W_w[0] = h / np.dot(h, h)                       # w_0 = +1, other heads 0
        q, w = l1_query(h, W_dq, W_iuq, W_w, n_h)
        K = (-np.abs(g.standard_normal((n, c_I))) * np.sign(q[0])[None, :]).astype(np.float32)   # q_0 . k < 0 everywhere
        hot = g.choice(n, size=3, replace=False)
        K[hot] = (4.0 * q[0] / np.dot(q[0], q[0])).astype(np.float32)                             # q_0 . k = 4
        planted |= {int(s) // C for s in hot}
        layers.append(dict(W_dq=W_dq, W_iuq=W_iuq, W_w=W_w))
        Ks.append(K)
    sel, val, cs, _ = l1_index_select(h, layers, Ks, n_h, C, k_max=16)
    got = {c for c in sel.tolist() if c >= 0}
    # unplanted entries have pre = 0 -> I = 0.5 -> recalled too (L4); planted ones rank first with sigmoid(4)
    assert planted.issubset(got)
    top = sel[: len(planted)].tolist()
    assert set(top) == planted and np.allclose(val[: len(planted)], 1 / (1 + np.exp(-4.0)), rtol=1e-5)
