"""Quality report on the ORACLE (SURVEY.md §5 "metrics", §8(d) config 5; "the pulses are not
flagged away", :164 flagged fraction): recall per injection class and false-positive rate for cut-down configs
2-5, and the on-pulse vs off-pulse flagged fraction of config 5.  Run `pytest tests/test_oracle_quality.py -s`
to see the table.  Gates are loose on purpose: under reading S4 (plain stddev, inflated by the RFI itself) weak
bursts are expected to be missed; the MAD scale (reading R1) is reported beside it."""
import numpy as np
import pytest

from paper_1701_08197_b200 import workloads as W

CLASS = {1: "narrow-band", 2: "spike", 3: "burst"}


def _report(lofo, name, power, truth, cls, C, T, mw, **kw):
    S = power.shape[0]
    rows = {}
    for mode, label in ((0, "stddev"), (1, "MAD")):
        prm = lofo.make_params(S, C, T, max_window=mw, stats_mode=mode, **kw)
        m = lofo.unpack_flags(lofo.flag_block_threads(prm, power, 8)["flags"], T).astype(bool)
        r = {"flagged": m.mean(), "false_pos": m[truth == 0].mean()}
        for k, nm in CLASS.items():
            sel = cls == k
            if sel.any():
                r[nm] = m[sel].mean()
        rows[label] = r
    print(f"\n{name}: " + "  ".join(f"[{lab}] " + " ".join(f"{k}={v:.3f}" for k, v in r.items()) for lab, r in rows.items()))
    return rows


def test_recall_per_class_config2(lofo):
    w = W.config2(0, n_stations=12)
    r = _report(lofo, "cfg2 (12 stations)", w.power, w.truth, w.extra["cls"], w.C, w.T, 64)
    # plain stddev (S4): the RFI inflates it 17-fold, events of 3-10 sigma stay under the thresholds (measured 0.67-0.72)
    assert min(r["stddev"][k] for k in CLASS.values()) > 0.5 and r["stddev"]["false_pos"] < 0.005
    # MAD scale (R1): everything injected is found, at 1.6 % false positives on Exp(1) noise (long tail)
    assert min(r["MAD"][k] for k in CLASS.values()) > 0.97 and r["MAD"]["false_pos"] < 0.03


def test_recall_per_class_config3(lofo):
    w = W.config3(0, n_stations=8)
    r = _report(lofo, "cfg3 (8 stations, 28 baselines)", w.power, w.truth, w.extra["cls"], w.C, w.T, 64)
    assert r["stddev"]["false_pos"] < 0.02                     # (recall 0.18-0.42: the stddev is inflated even more here)
    assert r["MAD"]["narrow-band"] > 0.95 and r["MAD"]["spike"] > 0.85 and r["MAD"]["false_pos"] < 0.02


def test_recall_per_class_config4(lofo):
    w = W.config4(0, n_stations=2, T=40000, want_truth=True)
    power = lofo.power_from_ci16(w.volt)
    r = _report(lofo, "cfg4 (2 stations, 40 000 samples)", power, w.truth, w.extra["cls"], w.C, w.T, 256)
    assert r["stddev"]["spike"] > 0.5 and r["stddev"]["false_pos"] < 0.02
    assert r["MAD"]["spike"] > 0.95 and r["MAD"]["burst"] > 0.9


def test_config5_pulse_is_not_flagged_away(lofo):
    """"the pulses are not flagged away".  Synthetic stand-in: a dispersed periodic pulse of +0.5 sigma
    that is NOT in the truth mask.  Measured on RFI-free samples: 2.5 % of the on-pulse samples are flagged against
    0.05 % off-pulse — in the RFI-free subbands the I = 64 level (1.07 sigma) is within reach of a 0.5-sigma excess
    488 samples wide — so the survey's tentative "on-pulse <= 2 x off-pulse" does not hold for this method; what does
    hold, and is gated here, is that the pulse survives: >= 95 % of its samples stay unflagged.  Also reported: the
    rate at which the history flagger (H = 300, literal 1-sigma threshold, reading H4') flags clean rows."""
    S, C, T = 12, 16, 12208
    gen = W.Config5Stream(0, S=S, C=C, T=T)
    kw = dict(max_window=64, history_length=300, history_min_fill=2)
    prm = lofo.make_params(S, C, T, **kw)
    hist = lofo.History(prm)
    on = off = n_on = n_off = 0
    rows_hist = rows_tot = rec = n_rfi = 0
    for k in range(6):
        w = gen.next_block()
        out = lofo.flag_block_threads(prm, w.power, 8)
        m = lofo.unpack_flags(out["flags"], T).astype(bool)
        clean = w.truth == 0
        p = w.extra["pulse"].astype(bool)
        on += m[clean & p].sum(); n_on += (clean & p).sum()
        off += m[clean & ~p].sum(); n_off += (clean & ~p).sum()
        rec += m[w.truth == 1].sum(); n_rfi += (w.truth == 1).sum()
        fl = out["flags"].copy()
        rf, _ = hist.update(out["rowsum"], out["rowcnt"], fl)
        clean_rows = w.truth.reshape(S * C, T).max(axis=1) == 0
        rows_hist += int(rf.reshape(-1)[clean_rows].sum()); rows_tot += int(clean_rows.sum())
    f_on, f_off = on / n_on, off / n_off
    print(f"\ncfg5 (12 subbands x 6 blocks): flagged on-pulse {f_on:.5f} off-pulse {f_off:.5f} ratio {f_on / max(f_off, 1e-12):.2f}; "
          f"narrow-band recall {rec / max(n_rfi, 1):.3f}; clean rows flagged by the history flagger {rows_hist}/{rows_tot}")
    assert n_on > 1000 and f_on < 0.05 and f_off < 0.002
    assert rec / max(n_rfi, 1) > 0.9
