"""Writes tests/golden/window_sha256.txt: the SHA-256 of every BASELINE.json config's window arrays (float64,
little-endian, W^TT | W^TP | W^PP) as paper_2602_15605_b200/windows.py draws them.  Calls windows.py only.

    python tests/golden/make_window_hashes.py

The test that reads the file (tests/test_windows_golden.py) makes a silent change of the inputs -- a different
numpy random stream, an edited recipe -- fail loudly: both arms of the bench, every rank and every parity test
must see these very inputs."""
import hashlib
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from paper_2602_15605_b200 import windows  # noqa: E402


def digest(wl):
    h = hashlib.sha256()
    for w in (wl.Wtt, wl.Wtp, wl.Wpp):
        if w is not None:
            h.update(w.astype("<f8").tobytes())
    return h.hexdigest()


def lines():
    out = ["# sha256 of the seeded window arrays of windows.config(i) (and of reduced-lmax variants the tests use)",
           "# written by tests/golden/make_window_hashes.py; columns: config lmax sha256"]
    for i in range(5):
        out.append("%d full %s" % (i, digest(windows.config(i))))
    for i, lm in ((1, 300), (2, 129), (1, 192)):
        out.append("%d %d %s" % (i, lm, digest(windows.config(i, lmax=lm))))
    return out


if __name__ == "__main__":
    with open(os.path.join(HERE, "window_sha256.txt"), "w") as fh:
        fh.write("\n".join(lines()) + "\n")
    print("\n".join(lines()))
