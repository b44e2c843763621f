"""Regenerates pin P14 of tests/golden/hand_example.json: eval losses of BASELINE.json configs 1
and 2 from the independent numpy-fp64 restatement tests/ref_numpy.py (NOT from the oracle under test and not
from the CUDA path), with the numpy recipes of datagen.py including numpy_init_weights (default_rng(2)).

    python tests/golden/make_p14.py            # print the block
    python tests/golden/make_p14.py --write    # rewrite the "P14" entry of hand_example.json

The stored values are rounded to 6 decimals, as SURVEY.md quotes them; config 2 takes ~1 minute."""
import json
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import ref_numpy as R                                   # noqa: E402
from paper_2606_30497_b200 import datagen               # noqa: E402


def block():
    out = {}
    c = datagen.CONFIGS["config1"]
    X, Y = datagen.make_dataset(c.n, c.sigma)
    W1, W2 = datagen.numpy_init_weights(c.hidden)
    w1, w2 = R.train(X, Y, W1, W2, c.batch, c.lr, c.epochs)
    out["config1"] = {"var_Y": round(float(np.var(Y.astype(np.float64))), 5),
                      "loss_init": round(R.eval_loss(X, Y, W1, W2), 6),
                      "loss_after_4_steps": round(R.eval_loss(X, Y, w1, w2), 6)}
    c = datagen.CONFIGS["config2"]
    X, Y = datagen.make_dataset(c.n, c.sigma)
    W1, W2 = datagen.numpy_init_weights(c.hidden)
    order = datagen.make_order(c.n, c.batch, c.epochs, c.shuffle)
    losses, w1, w2 = [], W1, W2
    for e in range(c.epochs):
        w1, w2 = R.train(X, Y, w1, w2, c.batch, c.lr, 1, order=order[e:e + 1])
        losses.append(round(R.eval_loss(X, Y, w1, w2), 6))
    out["config2"] = {"var_Y": round(float(np.var(Y.astype(np.float64))), 5),
                      "loss_init": round(R.eval_loss(X, Y, W1, W2), 6), "loss_after_epoch": losses}
    return out


if __name__ == "__main__":
    b = block()
    print(json.dumps(b, indent=1))
    if "--write" in sys.argv:
        path = os.path.join(HERE, "hand_example.json")
        d = json.load(open(path))
        b["_citation"] = d["P14"]["_citation"]
        d["P14"] = b
        json.dump(d, open(path, "w"), indent=1)
        print("rewrote", path)
