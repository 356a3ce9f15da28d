"""Asynchronous drain of the unweighted-event record buffer into an LHE 3.0 file ("The LHE writer ...
is run in a separate thread ... collects all the events ... and writes them (optionally compressed)").

Host policy and I/O only: the records are produced and compacted on the device by mf_unweight.  After an iteration

    drain.push(records, count, w_max)

enqueues, on a SIDE stream, the device->host copy of the cursor and of the filled part of the record buffer into
pinned memory, lets the compute stream wait only for that copy (so the next iteration may overwrite the buffer),
and hands the pinned block to a writer thread that formats and (optionally gzip-)writes the events while the GPU
computes the next iteration.  `close()` joins the thread and assembles header + events.

What the file contains: standard <init> and <event> blocks (IDWTUP = 3: unit weights, sign kept; overweight events
|w| > w_max keep |w| / w_max).  The records carry colour-SUMMED weights, so the colour flow written per event is one
fixed planar flow (t - g ... g - tbar in the order of the record), not a flow sampled from the colour-ordered
amplitudes; the header says so.
"""
import gzip
import io
import os
import queue
import threading

import numpy as np

PDG = {0: (11, -11, 13, -13), 1: (21, 21, 6, -6), 2: (21, 21, 6, -6, 21), 3: (21, 21, 6, -6, 21, 21),
       6: (21, 21, 6, -6, 21, 21, 21)}


QUARK_PDG = (1, 2, 3, 4, 5)          # flavour index of the multi-flavour table -> PDG id (d, u, s, c, b)


def record_dtype(n_final, process=None):
    fields = [("mom", np.float64, (n_final + 2, 4)), ("w", np.float64), ("id", np.uint64)]
    if process in (4, 5, 7):          # MF_PP_TT / MF_PP_TTG / MF_PP_TTGG records carry the partonic channel (include/mf.h)
        fields.append(("channel", np.uint64))
    return np.dtype(fields)


def channel_ids(channel):
    """PDG ids (beam 1, beam 2, t, tbar) and colour flow of an MF_PP_TT record's channel code"""
    c = int(channel)
    if c == 0:
        return PDG[1], colour_flow(1)
    q = QUARK_PDG[(c - 1) // 2]
    # q qbar -> g* -> t tbar: the quark's colour goes to the top, the antiquark's anticolour to the antitop
    if c % 2 == 1:
        return (q, -q, 6, -6), [(501, 0), (0, 502), (501, 0), (0, 502)]
    return (-q, q, 6, -6), [(0, 502), (501, 0), (501, 0), (0, 502)]


def channel_ids_ttj(channel):
    """PDG ids (beam 1, beam 2, t, tbar, parton) and one valid colour flow of an MF_PP_TTG record's channel code (R20):
    0 = gg; 1 + 6 i + c = flavour i in class c (q qbar, qbar q, q g, g q, qbar g, g qbar)"""
    c = int(channel)
    if c == 0:
        return PDG[2], colour_flow(2)
    q, cls = QUARK_PDG[(c - 1) // 6], (c - 1) % 6
    if cls < 2:          # q qbar -> t tbar g: q's colour to the gluon, the gluon's anticolour to the top, qbar's line to tbar
        ids, flow = [q, -q, 6, -6, 21], [(501, 0), (0, 502), (503, 0), (0, 502), (501, 503)]
    elif cls < 4:        # q g -> t tbar q: the quark line goes through; the gluon's colour to t, its anticolour to tbar
        ids, flow = [q, 21, 6, -6, q], [(501, 0), (502, 503), (502, 0), (0, 503), (501, 0)]
    else:                # qbar g -> t tbar qbar
        ids, flow = [-q, 21, 6, -6, -q], [(0, 501), (502, 503), (502, 0), (0, 503), (0, 501)]
    if cls & 1:          # the (anti)quark comes from beam 2
        ids[0], ids[1] = ids[1], ids[0]
        flow[0], flow[1] = flow[1], flow[0]
    return tuple(ids), flow


def channel_ids_ttgg(channel):
    """PDG ids (beam 1, beam 2, t, tbar, g, g) and one valid colour flow of an MF_PP_TTGG record's channel code (R22): 0 = gg;
    1 + 2 i = quark i from beam 1 and its antiquark from beam 2; 2 + 2 i = the other way round"""
    c = int(channel)
    if c == 0:
        return PDG[3], colour_flow(3)
    q = QUARK_PDG[(c - 1) // 2]
    # the quark's colour leaves on the first gluon, whose anticolour is the second gluon's colour, whose anticolour is the
    # top's colour; the antiquark's anticolour goes to the antitop
    ids, flow = [q, -q, 6, -6, 21, 21], [(501, 0), (0, 502), (504, 0), (0, 502), (501, 503), (503, 504)]
    if c % 2 == 0:
        ids[0], ids[1] = ids[1], ids[0]
        flow[0], flow[1] = flow[1], flow[0]
    return tuple(ids), flow


def colour_flow(process):
    """(colour, anticolour) tags per particle for the fixed planar flow; incoming gluons carry the crossed tags"""
    ids = PDG[process]
    if process == 0:
        return [(0, 0)] * 4
    # string: t (colour 501) - gluons in record order - tbar (anticolour = last tag)
    flow = [None] * len(ids)
    tag = 501
    flow[2] = (tag, 0)
    gluons = [i for i, p in enumerate(ids) if p == 21]
    for g in gluons:
        col, acol = tag + 1, tag            # an outgoing gluon absorbs `tag` as anticolour and emits tag + 1
        flow[g] = (acol, col) if g < 2 else (col, acol)    # crossed for the incoming ones
        tag += 1
    flow[3] = (0, tag)
    return flow


def format_events(rec, process, m_top, scale, alpha_em, alpha_s, w_max):
    """LHE <event> blocks for a structured record array (pure function: also used by the tests)"""
    per_event = process in (4, 5, 7)
    if not per_event:
        ids = PDG[process]
        flow = colour_flow(process)
    n = {4: 4, 5: 5, 7: 6}[process] if per_event else len(ids)
    out = io.StringIO()
    for r in rec:
        if per_event:
            ids, flow = {4: channel_ids, 5: channel_ids_ttj, 7: channel_ids_ttgg}[process](r["channel"])
        mass = [m_top if abs(p) == 6 else 0.0 for p in ids]
        w = float(r["w"])
        xw = (1.0 if w >= 0 else -1.0) * max(1.0, abs(w) / w_max)
        out.write("<event>\n%2d %d %+.10e %.10e %.10e %.10e\n" % (n, 1, xw, scale, alpha_em, alpha_s))
        for i in range(n):
            E, px, py, pz = r["mom"][i]
            ist, m1, m2 = (-1, 0, 0) if i < 2 else (1, 1, 2)
            out.write("%8d %2d %4d %4d %4d %4d %+.10e %+.10e %+.10e %.10e %.10e 0. 9.\n" %
                      (ids[i], ist, m1, m2, flow[i][0], flow[i][1], px, py, pz, E, mass[i]))
        out.write("# event id %d  weight %.10e pb\n</event>\n" % (int(r["id"]), w))
    return out.getvalue()


class LheDrain:
    def __init__(self, path, proc, compress=None):
        import torch
        if proc.wl.process not in PDG and proc.wl.process not in (4, 5, 7):
            raise ValueError("LHE output: unknown process %d" % proc.wl.process)
        self.torch = torch
        self.path = path
        self.proc = proc
        self.wl = proc.wl
        self.compress = path.endswith(".gz") if compress is None else compress
        self.dtype = record_dtype(proc.n_final, proc.wl.process)
        assert self.dtype.itemsize == proc.record_size
        self.side = torch.cuda.Stream()
        self.jobs = queue.Queue()
        # pinned staging buffers are allocated once and reused (cudaHostAlloc is slow and synchronising): the count, and a
        # ring of two record buffers that grow to the largest batch seen
        self._h_count = torch.empty(1, dtype=torch.int64).pin_memory()
        self._ring = [None, None]
        self._ring_free = [None, None]       # threading.Event: the writer thread has consumed the buffer
        self._turn = 0
        self.body_path = path + ".body"
        self.n_written = 0
        self.sum_w = 0.0
        self.error = None
        self.thread = threading.Thread(target=self._work, daemon=True)
        self.thread.start()

    # -- producer side (caller's thread) --------------------------------------------------------------------------
    def push(self, records, count, w_max, capacity, stream=None):
        """drain the records mf_unweight appended so far in `records` (uint8 CUDA tensor; cursor tensor `count`)"""
        torch = self.torch
        main = torch.cuda.current_stream() if stream is None else stream
        ready = torch.cuda.Event()
        ready.record(main)
        h_count = self._h_count
        with torch.cuda.stream(self.side):
            self.side.wait_event(ready)
            h_count.copy_(count, non_blocking=True)
            got_count = torch.cuda.Event()
            got_count.record(self.side)
        got_count.synchronize()                  # 8 bytes: the size of the next copy depends on it
        n = min(int(h_count.item()), capacity)
        nbytes = n * self.proc.record_size
        slot = self._turn
        self._turn ^= 1
        if self._ring_free[slot] is not None:
            self._ring_free[slot].wait()                      # the writer thread is done with this buffer
        if self._ring[slot] is None or self._ring[slot].numel() < max(nbytes, 1):
            self._ring[slot] = torch.empty(max(nbytes, 1 << 20), dtype=torch.uint8).pin_memory()
        h_rec = self._ring[slot]
        free = threading.Event()
        self._ring_free[slot] = free
        done = torch.cuda.Event()
        with torch.cuda.stream(self.side):
            if nbytes:
                h_rec[:nbytes].copy_(records[:nbytes], non_blocking=True)
            done.record(self.side)
        main.wait_event(done)                    # the buffer may be overwritten once the copy has run
        self.jobs.put((h_rec, n, done, float(w_max), free))
        return n

    # -- writer thread ---------------------------------------------------------------------------------------------
    def _work(self):
        try:
            opener = (lambda p: gzip.open(p, "wt")) if self.compress else (lambda p: open(p, "w"))
            with opener(self.body_path) as f:
                while True:
                    job = self.jobs.get()
                    if job is None:
                        break
                    h_rec, n, done, w_max, free = job
                    done.synchronize()
                    rec = np.frombuffer(h_rec.numpy()[:n * self.dtype.itemsize].tobytes(), dtype=self.dtype)   # a copy
                    free.set()                                # the staging buffer may be reused
                    rec = rec[np.argsort(rec["id"], kind="stable")]          # device order is unspecified
                    wl = self.wl
                    f.write(format_events(rec, wl.process, wl.m_top, np.sqrt(wl.mu2) if wl.process else wl.sqrt_s,
                                          wl.alpha_em, wl.alpha_s, w_max))
                    self.n_written += n
                    self.sum_w += float(rec["w"].sum())
        except Exception as e:      # reported by close()
            self.error = e

    def close(self, xsec_pb, xerr_pb):
        """joins the writer and assembles the file; xsec / error = the integration's combined estimate"""
        self.jobs.put(None)
        self.thread.join()
        if self.error is not None:
            raise self.error
        wl = self.wl
        beam = (11, -11) if wl.process == 0 else (2212, 2212)
        opener = (lambda p, m: gzip.open(p, m + "t")) if self.compress else (lambda p, m: open(p, m))
        with opener(self.path, "w") as f:
            f.write('<LesHouchesEvents version="3.0">\n<header>\n<!--\n')
            f.write("madflow-b200: %s, %d unweighted events (hit-or-miss against the running maximum weight)\n" %
                    (wl.name, self.n_written))
            f.write("colour flow: ONE fixed planar flow per partonic channel (the event weights are colour summed)\n")
            f.write("weights: IDWTUP = 3 with XWGTUP = sign(w); events with |w| > w_max (overweight) carry XWGTUP = sign(w) |w| / w_max > 1\n-->\n</header>\n")
            f.write("<init>\n%d %d %.8e %.8e 0 0 0 0 3 1\n%.10e %.10e 1.0 1\n</init>\n" %
                    (beam[0], beam[1], wl.sqrt_s / 2, wl.sqrt_s / 2, xsec_pb, xerr_pb))
            with opener(self.body_path, "r") as b:
                for line in b:
                    f.write(line)
            f.write("</LesHouchesEvents>\n")
        os.remove(self.body_path)
        return self.n_written
