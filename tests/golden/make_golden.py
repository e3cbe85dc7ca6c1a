"""Writes the stored expected values under tests/golden/.  Calls ONLY datagen/ and oracle/.

    python tests/golden/make_golden.py
"""
import hashlib
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import datagen  # noqa: E402


def main():
    w = datagen.make_weights(datagen.TINY)
    toks = datagen.tokens(1000, datagen.TINY.vocab, 32)
    out = {
        "tiny.embedding": hashlib.sha256(w.embedding.tobytes()).hexdigest(),
        "tiny.final_norm": hashlib.sha256(w.final_norm.tobytes()).hexdigest(),
        "tiny.l1.w_down": hashlib.sha256(w.layers[1]["w_down"].tobytes()).hexdigest(),
        "tiny.tokens32": toks.tolist(),
    }
    with open(os.path.join(HERE, "datagen_checksums.json"), "w") as f:
        json.dump(out, f, indent=1)
        f.write("\n")


if __name__ == "__main__":
    main()
