"""LHE 3.0 output of the unweighted events: the pure formatting functions on CPU,
the asynchronous drain on the GPU."""
import gzip
import re

import numpy as np
import pytest

from paper_2106_10279_b200 import lhe
from paper_2106_10279_b200 import workloads as W


def _parse(text):
    events = []
    for blk in re.findall(r"<event>\n(.*?)</event>", text, re.S):
        lines = [l for l in blk.strip().split("\n") if not l.startswith("#")]
        head = lines[0].split()
        parts = [l.split() for l in lines[1:]]
        eid = int(re.search(r"# event id (\d+)", blk).group(1))
        events.append((int(head[0]), float(head[2]), parts, eid))
    return events


def test_colour_flow_is_a_valid_planar_flow():
    for proc in (1, 2, 3):
        ids, flow = lhe.PDG[proc], lhe.colour_flow(proc)
        out_col, out_acol = [], []
        for i, (pid, (c, a)) in enumerate(zip(ids, flow)):
            if i < 2:                       # incoming: crossing swaps the roles
                c, a = a, c
            if c:
                out_col.append(c)
            if a:
                out_acol.append(a)
            assert (pid == 21) == (c != 0 and a != 0)
        assert sorted(out_col) == sorted(out_acol)           # every colour line ends on an anticolour
        assert len(set(out_col)) == len(out_col)


def test_format_events_round_trip():
    rng = np.random.default_rng(0)
    rec = np.zeros(5, dtype=lhe.record_dtype(4))
    rec["mom"] = rng.normal(size=(5, 6, 4)) * 300
    rec["w"] = [1.0, -0.5, 3.0, 2.0, 0.25]
    rec["id"] = [7, 3, 2 ** 40 + 1, 11, 5]
    text = lhe.format_events(rec, 3, 173.0, 173.0, 1 / 132.507, 0.118, w_max=2.0)
    ev = _parse(text)
    assert len(ev) == 5 and [e[3] for e in ev] == [7, 3, 2 ** 40 + 1, 11, 5]
    assert [e[1] for e in ev] == [1.0, -1.0, 1.5, 1.0, 1.0]          # unit weights, sign kept, overweight 3/2
    for (nup, _, parts, _), r in zip(ev, rec):
        assert nup == 6 and [int(p[0]) for p in parts] == [21, 21, 6, -6, 21, 21]
        assert [int(p[1]) for p in parts] == [-1, -1, 1, 1, 1, 1]
        for p, m in zip(parts, r["mom"]):
            got = np.array([float(p[9]), float(p[6]), float(p[7]), float(p[8])])     # E px py pz
            np.testing.assert_allclose(got, m, rtol=2e-10, atol=1e-9)
        assert [float(p[10]) for p in parts] == [0, 0, 173, 173, 0, 0]


def test_flavour_summed_records_carry_their_partons():
    """MF_PP_TT: PDG ids and colour flow follow the channel code of each record (include/mf.h)"""
    rec = np.zeros(4, dtype=lhe.record_dtype(2, 4))
    assert rec.dtype.itemsize == 4 * 32 + 24
    rec["channel"] = [0, 1, 4, 7]
    rec["w"] = 1.0
    ev = _parse(lhe.format_events(rec, 4, 173.0, 173.0, 1 / 132.507, 0.118, w_max=1.0))
    assert [[int(p[0]) for p in e[2]] for e in ev] == [[21, 21, 6, -6], [1, -1, 6, -6], [-2, 2, 6, -6], [4, -4, 6, -6]]
    for _, _, parts, _ in ev:
        col_in = sorted(int(p[4]) for p in parts[:2] if int(p[4]))
        acol_in = sorted(int(p[5]) for p in parts[:2] if int(p[5]))
        col_out = sorted(int(p[4]) for p in parts[2:] if int(p[4]))
        acol_out = sorted(int(p[5]) for p in parts[2:] if int(p[5]))
        for p in parts:             # quarks carry a colour, antiquarks an anticolour, gluons both
            pid, c, a = int(p[0]), int(p[4]), int(p[5])
            assert (c != 0) == (pid == 21 or pid > 0) and (a != 0) == (pid == 21 or pid < 0)
        # colour is conserved: what flows in and does not annihilate flows out
        assert sorted(set(col_in) - set(acol_in)) == col_out and sorted(set(acol_in) - set(col_in)) == acol_out


def test_ttj_records_carry_their_partons():
    """MF_PP_TTG (R20): PDG ids and a colour-conserving flow for every class and beam assignment"""
    rec = np.zeros(7, dtype=lhe.record_dtype(3, 5))
    assert rec.dtype.itemsize == 5 * 32 + 24
    rec["channel"] = [0, 1, 2, 1 + 6 + 2, 1 + 6 + 3, 1 + 12 + 4, 1 + 18 + 5]
    rec["w"] = 1.0
    ev = _parse(lhe.format_events(rec, 5, 173.0, 173.0, 1 / 132.507, 0.118, w_max=1.0))
    assert [[int(p[0]) for p in e[2]] for e in ev] == [[21, 21, 6, -6, 21], [1, -1, 6, -6, 21], [-1, 1, 6, -6, 21],
                                                       [2, 21, 6, -6, 2], [21, 2, 6, -6, 2], [-3, 21, 6, -6, -3],
                                                       [21, -4, 6, -6, -4]]
    for _, _, parts, _ in ev:
        col_in = sorted(int(p[4]) for p in parts[:2] if int(p[4]))
        acol_in = sorted(int(p[5]) for p in parts[:2] if int(p[5]))
        col_out = sorted(int(p[4]) for p in parts[2:] if int(p[4]))
        acol_out = sorted(int(p[5]) for p in parts[2:] if int(p[5]))
        for p in parts:
            pid, c, a = int(p[0]), int(p[4]), int(p[5])
            assert (c != 0) == (pid == 21 or pid > 0) and (a != 0) == (pid == 21 or pid < 0)
        # colour conservation: incoming colours = outgoing colours up to lines created in pairs (colour + anticolour out)
        created = set(col_out) & set(acol_out)
        assert sorted(set(col_in) - set(acol_in)) == sorted(set(col_out) - created)
        assert sorted(set(acol_in) - set(col_in)) == sorted(set(acol_out) - created)


def test_ttgg_records_carry_their_partons():
    """MF_PP_TTGG (R22): gg or q qbar of the record's flavour, the quark from either beam, with a colour-conserving flow"""
    rec = np.zeros(5, dtype=lhe.record_dtype(4, 7))
    assert rec.dtype.itemsize == 6 * 32 + 24
    rec["channel"] = [0, 1, 2, 5, 8]
    rec["w"] = 1.0
    ev = _parse(lhe.format_events(rec, 7, 173.0, 173.0, 1 / 132.507, 0.118, w_max=1.0))
    assert [[int(p[0]) for p in e[2]] for e in ev] == [[21, 21, 6, -6, 21, 21], [1, -1, 6, -6, 21, 21], [-1, 1, 6, -6, 21, 21],
                                                       [3, -3, 6, -6, 21, 21], [-4, 4, 6, -6, 21, 21]]
    for _, _, parts, _ in ev:
        col_in = sorted(int(p[4]) for p in parts[:2] if int(p[4]))
        acol_in = sorted(int(p[5]) for p in parts[:2] if int(p[5]))
        col_out = sorted(int(p[4]) for p in parts[2:] if int(p[4]))
        acol_out = sorted(int(p[5]) for p in parts[2:] if int(p[5]))
        for p in parts:
            pid, c, a = int(p[0]), int(p[4]), int(p[5])
            assert (c != 0) == (pid == 21 or pid > 0) and (a != 0) == (pid == 21 or pid < 0)
        created = set(col_out) & set(acol_out)
        assert sorted(set(col_in) - set(acol_in)) == sorted(set(col_out) - created)
        assert sorted(set(acol_in) - set(col_in)) == sorted(set(acol_out) - created)


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,n_ev,div,ids_of,nup_want", [("C5", 30000, 30, "channel_ids", 4), ("C6", 30000, 30, "channel_ids_ttj", 5),
                                                         ("C8", 20000, 300, "channel_ids_ttgg", 6)])
def test_lhe_drain_flavour_summed(tmp_path, cfg, n_ev, div, ids_of, nup_want):
    """the drain on MF_PP_TT / MF_PP_TTG / MF_PP_TTGG records: every event of the file has the partons of its record's channel"""
    import torch
    from paper_2106_10279_b200 import api
    wl = {"C5": W.C5, "C6": W.C6, "C8": W.C8}[cfg].scaled(n_ev, 2, 1)
    gp = api.Process(wl, W.pdf_table_flavours())
    grid, hist, res = gp.new_grid(), gp.new_hist(), gp.new_result()
    gp.vegas_iterate(grid, 0, 0, 0, wl.n_events, hist, res)
    gp.refine_grid(grid, hist)
    w_max = gp.result_to_host(res).max_abs_w / div
    cap = n_ev
    records = torch.zeros(cap * gp.record_size, dtype=torch.uint8, device="cuda")
    count = torch.zeros(1, dtype=torch.int64, device="cuda")
    path = str(tmp_path / "pp.lhe")
    drain = lhe.LheDrain(path, gp)
    gp.unweight(grid, 0, 1, 0, wl.n_events, w_max, records, cap, count, None, res)
    n = drain.push(records, count, w_max, cap)
    torch.cuda.synchronize()
    mom, w, ids = gp.records_view(records, n)
    chan = gp.records_array(records, n)["channel"][np.argsort(ids)]
    assert drain.close(2760.0, 0.4) == n and n > 100 and (chan > 0).sum() > 5
    ev = _parse(open(path).read())
    assert len(ev) == n
    for (nup, _, parts, _), c in zip(ev, chan):
        want, _ = getattr(lhe, ids_of)(c)
        assert nup == nup_want and tuple(int(p[0]) for p in parts) == tuple(want)
    gp.close()


@pytest.mark.gpu
@pytest.mark.parametrize("compress", [False, True])
def test_lhe_drain_matches_records(tmp_path, compress, pdf):
    """frozen iterations of gg -> ttbar with unweighting, each drained asynchronously: the file holds exactly the
    accepted events of every iteration, in event-id order per iteration, momenta to the printed precision"""
    import torch
    from paper_2106_10279_b200 import api
    wl = W.C1.scaled(30000, 4, 2)
    gp = api.Process(wl, pdf)
    grid, hist, res = gp.new_grid(), gp.new_hist(), gp.new_result()
    w_max = 0.0
    for k in range(2):
        gp.vegas_iterate(grid, 0, k, 0, wl.n_events, hist, res)
        gp.refine_grid(grid, hist)
        w_max = max(w_max, gp.result_to_host(res).max_abs_w)
    cap = 4096
    records = torch.zeros(cap * gp.record_size, dtype=torch.uint8, device="cuda")
    count = torch.zeros(1, dtype=torch.int64, device="cuda")
    path = str(tmp_path / ("ev.lhe.gz" if compress else "ev.lhe"))
    drain = lhe.LheDrain(path, gp)
    want = []
    for k in range(2, 4):
        count.zero_()
        gp.unweight(grid, 0, k, 0, wl.n_events, w_max, records, cap, count, None, res)
        n = drain.push(records, count, w_max, cap)
        torch.cuda.synchronize()
        mom, w, ids = gp.records_view(records, n)
        order = np.argsort(ids)
        want += [(int(ids[i]), mom[i].copy(), float(w[i])) for i in order]
        assert n == gp.result_to_host(res).n_accept > 0
    n_tot = drain.close(2649.0, 0.4)
    text = (gzip.open(path, "rt") if compress else open(path)).read()
    assert text.startswith('<LesHouchesEvents version="3.0">') and text.rstrip().endswith("</LesHouchesEvents>")
    assert re.search(r"<init>\n2212 2212 6\.5", text)
    ev = _parse(text)
    assert len(ev) == n_tot == len(want)
    for (nup, xw, parts, eid), (wid, wm, ww) in zip(ev, want):
        assert eid == wid and nup == 4 and xw == (1.0 if ww >= 0 else -1.0) * max(1.0, abs(ww) / w_max)
        for p, m in zip(parts, wm):
            np.testing.assert_allclose([float(p[9]), float(p[6]), float(p[7]), float(p[8])], m, rtol=2e-10, atol=1e-8)
    gp.close()
