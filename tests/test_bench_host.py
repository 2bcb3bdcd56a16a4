"""Host-side logic of bench.py that needs no GPU: the summary of a per-CTA timeline (include/lsa.h LSA_TL_*)."""
import importlib.util
import os

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _bench():
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(ROOT, "bench.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def test_summarise_timeline_on_a_constructed_ring():
    """Two launches of 4 CTAs on 2 SMs, the last 2 arrivals of each merge: every figure of the summary follows by hand."""
    b = _bench()
    ENTRY, SETUP, FIRST_S, LAST_PV, EPI, ARRIVED, ALL_ARR, MERGED, EXIT, SMID, NCTAS, SEQ = range(12)
    rec = np.zeros((16, 160, 12), dtype=np.uint64)
    t0 = 1_000_000
    for l in range(2):
        for cta in range(4):
            e = t0 + l * 40_000 + (cta // 2) * 20_000           # two CTAs at a time, one after the other on each SM
            r = rec[l, cta]
            r[ENTRY], r[SETUP], r[FIRST_S], r[LAST_PV], r[EPI], r[ARRIVED] = e, e + 2000, e + 4000, e + 12000, e + 13000, e + 15000
            if cta >= 2:                                         # mergers: wait 1 us, merge 3 us
                r[ALL_ARR], r[MERGED], r[EXIT] = e + 16000, e + 19000, e + 19500
            else:
                r[EXIT] = e + 15500
            r[SMID], r[NCTAS], r[SEQ] = cta % 2, 4, l
    rec[3, 0, NCTAS] = 4                                         # a record that was being overwritten: exit <= entry, dropped
    s = b.summarise_timeline([rec], step_ms=0.02)
    assert s["launches"] == 2 and s["ctas_per_launch"] == 4 and s["mergers_per_launch"] == 2 and s["sms_seen"] == 2
    a = s["all_ctas_us"]
    assert a["entry_to_setup"] == 2.0 and a["entry_to_first_s"] == 4.0 and a["first_s_to_last_pv"] == 8.0
    assert a["last_pv_to_epilogue"] == 1.0 and a["epilogue_to_arrived"] == 2.0
    assert s["leavers_us"]["residence"] == 15.5
    assert s["mergers_us"] == dict(arrived_to_all_arrived=1.0, all_arrived_to_merged=3.0, residence=19.5)
    assert s["sm_residence_us_per_launch"] == 2 * 15.5 + 2 * 19.5
    # hand-overs on an SM: leaver (exit e + 15.5) -> merger (entry e + 20): 4.5 us; merger (exit e + 39.5) -> next launch (e + 40): 0.5 us
    assert s["handover_us_median"] in (0.5, 2.5, 4.5)
    assert abs(s["step_us_if_sm_bound"] - (70.0 + 4 * s["handover_us_median"]) / 148.0) < 1e-9
    assert b.summarise_timeline([np.zeros((16, 160, 12), dtype=np.uint64)], 0.01) is None
