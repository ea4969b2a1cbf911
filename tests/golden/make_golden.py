"""Writes tests/golden/cfg1_oracle.txt: oracle SNR at 12 fixed (k, x, y) of config 1.
Calls only oracle/ and tno_synth/ (never the CUDA path).  Run: python tests/golden/make_golden.py
"""
import os
import sys

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "..", ".."))
import oracle          # noqa: E402
import tno_synth       # noqa: E402


def main():
    p = tno_synth.make_params(tno_synth.CONFIGS[1])
    f = tno_synth.stack_numpy(p)
    oracle.inject(f, p.traj[p.src_k], p.src_x, p.src_y, p.src_amp, p.cfg.prf_sigma, p.cfg.t0)
    pts = [(int(p.src_k[i]), int(p.src_x[i]), int(p.src_y[i])) for i in range(len(p.src_k))]
    pts += [(k, x, y) for k, x, y in ((0, 0, 0), (4, 63, 63), (8, 0, 63), (2, 31, 0), (6, 17, 40),
                                       (1, 1, 1), (3, 62, 5), (5, 33, 33), (7, 5, 60), (4, 20, 20))]
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg1_oracle.txt")
    with open(out, "w") as fh:
        fh.write("# written by tests/golden/make_golden.py (oracle/ + tno_synth/ only)\n")
        fh.write("# config 1 of BASELINE.json, sources injected with oracle.inject\n# k x y snr\n")
        for k, x, y in pts:
            s, _, _ = oracle.point(f, p.sigma_t, p.traj[k], p.cfg.prf_sigma, p.cfg.t0, x, y)
            fh.write("%d %d %d %.17g\n" % (k, x, y, s))
    print("wrote", out)


if __name__ == "__main__":
    main()
