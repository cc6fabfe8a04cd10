"""How far the canonical-fp32 pipeline (O32, the parity target) sits from the same method evaluated in fp64 throughout
(O64) -- SURVEY 8(c) "Oracle variants".  Calls only oracle/ and the input generators.  TEST INFRASTRUCTURE.

    python -m oracle.o64_report [--config1]      # markdown table on stdout (committed as profiles/r2_o64_report.md)

Rect differences are expected: O32's rect is the PADDED box (h (1 + 2^-10) + 2^-6, DESIGN O4) of the contour, O64's the
exact one, so O32 may hold a few more tiles; what matters is that O64's rect never sticks out of O32's (conservative)."""
import sys

import numpy as np

import flod_synth as fs
from oracle import OracleScene, ST_VISIBLE


def compare(osc, cam, ls, le, gamma, label, image=True):
    a = osc.frame(cam, ls, le, gamma, geometry_only=not image)
    b = osc.frame(cam, ls, le, gamma, geometry_only=not image, fp64=True)
    ra, rb = a.rect, b.rect
    both = (a.state == ST_VISIBLE) & (b.state == ST_VISIBLE)
    sticks_out = both & ((rb[:, 0] < ra[:, 0]) | (rb[:, 1] < ra[:, 1]) | (rb[:, 2] > ra[:, 2]) | (rb[:, 3] > ra[:, 3]))
    row = [label, a.counts["n_sel"], int((a.mask != b.mask).sum()), a.counts["n_vis"], int((a.state != b.state).sum()),
           int((ra != rb).any(axis=1)[both].sum()), int(sticks_out.sum()), a.counts["n_pairs"], b.counts["n_pairs"]]
    if image:
        d = np.abs(a.composite() - b.composite())
        row += [f"{d.max():.2e}", f"{np.quantile(d, 0.999):.2e}", int((d.max(axis=0) > 1e-3).sum())]
    else:
        row += ["-", "-", "-"]
    return row


def main():
    rows = []
    sc = fs.make_scene(0)
    cam = fs.make_poses(0)[0]
    osc = OracleScene(sc.levels, sc.sh_degree)
    rows.append(compare(osc, cam, 2, 2, 1.0, "config 0, level 2"))
    rows.append(compare(osc, cam, 1, 2, 1.0, "config 0, {1,2} gamma 1"))
    if "--config1" in sys.argv:
        sc = fs.make_scene(1)
        cams = fs.make_poses(1)
        osc = OracleScene(sc.levels, sc.sh_degree)
        rows.append(compare(osc, cams[0], 5, 5, 1.0, "config 1, level 5, pose 0"))
        rows.append(compare(osc, cams[0], 3, 5, 1.0, "config 2, {3,4,5} gamma 1, pose 0"))
        rows.append(compare(osc, cams[0], 3, 5, 4.0, "config 2, {3,4,5} gamma 4, pose 0"))
    head = ["frame", "N_sel", "mask bits that differ", "N_vis", "cull states that differ", "rects that differ",
            "O64 rect outside O32 rect", "P (O32)", "P (O64)", "max abs image diff", "99.9 % quantile", "pixels > 1e-3"]
    print("| " + " | ".join(head) + " |")
    print("|" + "---|" * len(head))
    for r in rows:
        print("| " + " | ".join(str(x) for x in r) + " |")


if __name__ == "__main__":
    main()
