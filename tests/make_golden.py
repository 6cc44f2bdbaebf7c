"""Writes tests/golden/e1_stream.hex from docs/FORMAT.md via tests/streams.py (pure Python only)."""
import os
from streams import build_stream

E1 = [[(b"abcdefgh", 8, 0), (b"WX", 8, 0), (b"z", 5, 26)]]
if __name__ == "__main__":
    s = build_stream(E1, 32, flags=5)
    here = os.path.dirname(os.path.abspath(__file__))
    with open(os.path.join(here, "golden", "e1_stream.hex"), "w") as f:
        f.write("# docs/FORMAT.md layout of example E1, flatten on; written by tests/make_golden.py\n")
        h = s.tobytes().hex()
        for i in range(0, len(h), 64):
            f.write(h[i:i + 64] + "\n")
