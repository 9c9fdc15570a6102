"""Reader for tests/golden/paper_values.txt (values the paper prints, each with its citation)."""
import os


def load():
    out = {}
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_values.txt")
    with open(path) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            toks = line.split()
            key, vals = toks[0], []
            for t in toks[1:]:
                try:
                    vals.append(float(t))
                except ValueError:
                    break
            out[key] = vals[0] if len(vals) == 1 else vals
    return out
