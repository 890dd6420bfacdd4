"""Reader for the `key: v1, v2, ...` fixtures in tests/golden/ (see tests/golden/README.md)."""
import os


def load(name):
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", name)) as fh:
        for line in fh:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            key, _, val = line.partition(":")
            items = [v.strip() for v in val.split(",")]
            try:
                out[key.strip()] = [float(v) for v in items]
            except ValueError:
                out[key.strip()] = items
    return out
