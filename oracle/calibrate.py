"""Writes gen/calib.json: per (config k, T) the gains of the synthetic-weights recipe.

  wc[t] : factor on Wc[t]            so that rms(rho^t)   ~ 1
  c[t]  : factor on the last layer of coefficient network t   so that rms(c^{t+1}) ~ 1
  e     : factor on the last layer of the energy network      so that rms|F| ~ 1 eV/A

Without them the random networks collapse onto their biases after the first layer and the
message-passing terms of the backward pass would sit below the parity tolerance. Measured
layer by layer with the ORACLE ONLY (never the CUDA path) on same-density replicas
(216 H2O / 6^3 fcc cells) built with the same seeds. Run:  python oracle/calibrate.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import gen          # noqa: E402
import oracle       # noqa: E402


def rms(x):
    return float(np.sqrt((x ** 2).mean()))


def calibrate(k, T, kw):
    T = gen.CONFIGS[k]["T"] if T is None else T
    g = dict(wc=[1.0] * T, c=[1.0] * (T - 1), e=1.0)

    def run(forces=False):
        cfg = gen.make_config(k, T=T, gains=g, **kw)
        return oracle.energy_forces(cfg["blob"], cfg["species"], cfg["pos"], cfg["box"], forces=forces, dumps=True)
    for t in range(T):
        g["wc"][t] = 1.0 / np.sqrt(rms(run()["rho"][t]))        # rho is quadratic in Wc
        if t < T - 1:
            g["c"][t] = 1.0 / rms(run()["c"][t + 1])
    r = run(True)
    g["e"] = 1.0 / float(np.sqrt((r["F"] ** 2).sum(1).mean()))
    g = dict(wc=[round(x, 6) for x in g["wc"]], c=[round(x, 6) for x in g["c"]], e=round(g["e"], 6))
    return g


def main():
    table = {}
    jobs = [(0, None), (1, None), (2, None), (3, None), (5, None)] + [(4, T) for T in range(1, 7)]
    for k, T in jobs:
        kw = {}
        if k in (2, 3, 5):
            kw["n_mol"] = 216
        if k == 4:
            kw["ncell"] = 6
        g = calibrate(k, T, kw)
        cfg = gen.make_config(k, T=T, gains=g, **kw)
        r = oracle.energy_forces(cfg["blob"], cfg["species"], cfg["pos"], cfg["box"], dumps=True)
        table[f"{k}:{cfg['T']}"] = g
        print(k, cfg["T"], g, "-> rms|F| %.4f" % np.sqrt((r["F"] ** 2).sum(1).mean()),
              "rho rms", [round(rms(x), 3) for x in r["rho"]], "c rms", [round(rms(x), 3) for x in r["c"]],
              "c std/atoms", [round(float(x.std(0).mean()), 3) for x in r["c"]])
    with open(os.path.join(ROOT, "gen", "calib.json"), "w") as f:
        json.dump(table, f, indent=1, sort_keys=True)


if __name__ == "__main__":
    main()
