"""Re-derive tests/golden/p15_*.txt from the oracle side only (oracle/mp_chain.py,
mpmath at 50 digits, §3.2) and report the difference from the stored
(survey-computed) values. Usage: python tests/golden/make_golden.py [--write]
With --write the files' data rows are rewritten from mp_chain (headers kept).
Calls nothing outside oracle/ and dfr_synth (input recipe)."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import mpmath as mp  # noqa: E402

import dfr_synth as S  # noqa: E402
from oracle import mp_chain  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))


def rows(path):
    head, data = [], []
    for line in open(path):
        (head if line.startswith("#") else data).append(line.rstrip("\n"))
    return head, [d.split() for d in data if d.strip()]


def main(write):
    w0 = S.config0()
    src, tgt = w0.src_wcs[0], w0.tgt_wcs
    path = os.path.join(HERE, "p15_config0_pair.txt")
    head, data = rows(path)
    out, worst = [], 0.0
    for r in data:
        tx, ty = mp.mpf(r[0]), mp.mpf(r[1])
        ra, dec = mp_chain.pix2world_deg(tgt, tx, ty)
        new = [r[0], r[1], mp.nstr(ra, 17), mp.nstr(dec, 17)]
        worst = max(worst, abs(float(ra) - float(r[2])), abs(float(dec) - float(r[3])))
        if r[4] != "-":
            x, y = mp_chain.src_coord(tgt, src, tx, ty)
            new += [mp.nstr(x, 15), mp.nstr(y, 15)]
            worst = max(worst, abs(float(x) - float(r[4])), abs(float(y) - float(r[5])))
        else:
            new += ["-", "-"]
        out.append(" ".join(new))
    print("p15_config0_pair: max |mp_chain - stored| =", worst)
    if write:
        open(path, "w").write("\n".join(head + out) + "\n")

    w = S.make_wcs(2048, 2048, 210.25, -35.5, 0.5, S.PIXSCALE)
    w.a[2, 0], w.a[1, 1], w.a[0, 3] = 2e-6, -1e-6, 3e-10
    w.b[0, 2], w.b[2, 1] = -1.5e-6, 2e-10
    w.a_order = w.b_order = 3
    path = os.path.join(HERE, "p15_sip_example.txt")
    head, data = rows(path)
    out, worst = [], 0.0
    for r in data:
        ra, dec = mp_chain.pix2world_deg(w, mp.mpf(r[0]), mp.mpf(r[1]))
        worst = max(worst, abs(float(ra) - float(r[2])), abs(float(dec) - float(r[3])))
        out.append(" ".join([r[0], r[1], mp.nstr(ra, 17), mp.nstr(dec, 17)]))
    print("p15_sip_example: max |mp_chain - stored| =", worst)
    if write:
        open(path, "w").write("\n".join(head + out) + "\n")


if __name__ == "__main__":
    main("--write" in sys.argv)
