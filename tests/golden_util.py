"""Reader for tests/golden/*.txt fixtures (key = value  # citation)."""
import os


def load(name="closed_forms.txt"):
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)
    out = {}
    with open(path) as fh:
        for line in fh:
            line = line.split("#", 1)[0].strip()
            if not line:
                continue
            k, v = line.split("=", 1)
            out[k.strip()] = float(v)
    return out
