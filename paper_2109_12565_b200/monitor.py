"""Run-time Delaunay monitor (host logic only; every analysis step is a call of the C ABI, include/tlb.h).

The paper's workflow (Table C.12): every `ncheckdelaunay` steps the droplets are identified, triangulated
and compared with the previous frame; frames with T1 events go to ./delaunayTriggerDir, the others to
./delaunayNoTriggerDir, together with the time sequences nBubblesOut / nLinksOut and the lists breakingLinks /
arisingLinks.  The paper names the files and defers their structure to its sources; reading R32:

  nBubblesOut, nLinksOut          ASCII, one line "step value" per check
  breakingLinks, arisingLinks     ASCII, one line "step a b" per T1 event: the link that vanished / appeared, in the
                                  droplet indices of the PAST frame (rank in ascending label order)
  delaunayNowTime<step>,          little-endian binary frame: int32 n_droplets, int32 n_links,
  delaunayPastTime<step>          float64 centres[n_droplets][2] (x, y), int32 links[n_links][2] (a < b, sorted)

This module holds none of the method's arithmetic and never imports anything under oracle/.
"""
import os

import numpy as np


class Frame:
    """Centres, Voronoi colouring and links of one instant (device tensors) + the step it was taken at."""

    def __init__(self, step, n, centres, colour, links):
        self.step, self.n, self.centres, self.colour, self.links = step, n, centres, colour, links

    def tofile(self, path):
        with open(path, "wb") as f:
            np.array([self.n, int(self.links.shape[0])], dtype="<i4").tofile(f)
            self.centres.cpu().numpy().astype("<f8").tofile(f)
            self.links.cpu().numpy().astype("<i4").tofile(f)


def read_frame(path):
    """(centres [n][2] float64, links [m][2] int32) of a frame file written by Frame.tofile."""
    with open(path, "rb") as f:
        n, m = np.fromfile(f, dtype="<i4", count=2)
        centres = np.fromfile(f, dtype="<f8", count=2 * n).reshape(n, 2)
        links = np.fromfile(f, dtype="<i4", count=2 * m).reshape(m, 2)
    return centres, links


class DelaunayMonitor:
    def __init__(self, tlb, B_th, out_dir, max_droplets=4096, max_events=4096):
        self.t, self.B_th, self.dir = tlb, float(B_th), out_dir
        self.max_droplets, self.max_events = int(max_droplets), int(max_events)
        self.trig = os.path.join(out_dir, "delaunayTriggerDir")
        self.notrig = os.path.join(out_dir, "delaunayNoTriggerDir")
        os.makedirs(self.trig, exist_ok=True)
        os.makedirs(self.notrig, exist_ok=True)
        self.past = None

    def frame(self, step):
        """tlb_droplets -> tlb_voronoi -> tlb_delaunay on the current state."""
        _, k, stats = self.t.droplets(self.B_th, self.max_droplets, want_labels=False)
        if k > self.max_droplets:
            raise ValueError("%d droplets exceed max_droplets = %d" % (k, self.max_droplets))
        centres = stats[:, 2:4].contiguous()
        colour = self.t.voronoi(centres)
        links, nl = self.t.delaunay(colour, k, max_links=16 * max(k, 1))
        if nl < 0:
            raise ValueError("a droplet has more links than the adjacency table holds")
        return Frame(step, k, centres, colour, links)

    def compare(self, past, now):
        """(events [e][4], displacements [n_now][2], map [n_now]) between two frames: tlb_droplet_match, tlb_t1_events,
        tlb_droplet_displacements."""
        mp = self.t.droplet_match(past.colour, now.centres)
        ev, ne = self.t.t1_events(past.links, now.links, past.n, mp, max_events=self.max_events)
        if ne < 0 or ne > self.max_events:
            raise ValueError("T1 event table overflow")
        disp = self.t.droplet_displacements(past.centres, now.centres, mp)
        return ev, disp, mp

    def _append(self, name, line, directory=None):
        with open(os.path.join(directory or self.dir, name), "a") as f:
            f.write(line)

    def record(self, now):
        """Compare `now` with the stored past frame, write the files of Table C.12, keep `now` as the next past frame.
        Returns the events as an int array [e][4] (empty for the first frame)."""
        self._append("nBubblesOut", "%d %d\n" % (now.step, now.n))
        self._append("nLinksOut", "%d %d\n" % (now.step, int(now.links.shape[0])))
        events = np.zeros((0, 4), dtype=np.int32)
        if self.past is not None:
            ev, _, _ = self.compare(self.past, now)
            events = ev.cpu().numpy()
        if len(events):
            for a, b, c, d in events:
                self._append("breakingLinks", "%d %d %d\n" % (now.step, a, b), self.trig)
                self._append("arisingLinks", "%d %d %d\n" % (now.step, c, d), self.trig)
            self.past.tofile(os.path.join(self.trig, "delaunayPastTime%d" % now.step))
            now.tofile(os.path.join(self.trig, "delaunayNowTime%d" % now.step))
        else:
            now.tofile(os.path.join(self.notrig, "delaunayNowTime%d" % now.step))
        self.past = now
        return events

    def check(self, step):
        """One run-time check at `step` (the paper's ncheckdelaunay cadence is the caller's loop)."""
        return self.record(self.frame(step))
