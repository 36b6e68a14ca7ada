"""reader for the small 'key = v v v' text fixtures under tests/golden/."""
import os

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def load(name):
    out = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, v = line.split("=", 1)
            toks = v.split()
            try:
                out[k.strip()] = [int(t) for t in toks]
            except ValueError:
                out[k.strip()] = v.strip()
    return out
