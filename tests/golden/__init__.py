"""Golden values: paper_constants.txt holds numbers printed in the paper, each with its PAPER.md citation."""
import os


def load_paper_constants():
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "paper_constants.txt")) as fh:
        for line in fh:
            line = line.split("#")[0].strip()
            if not line:
                continue
            key, val = [t.strip() for t in line.split("=")]
            out[key] = [float(t) if ("e" in t or "." in t) else int(t) for t in val.split()]
    return out
