"""Build the CPU oracle (TEST INFRASTRUCTURE) twice from oracle/lisa_oracle.c.

  liboracle_f64.so : real = double       (timed cpu_baseline, fp64 noise floor)
  liboracle_f80.so : real = long double  (the parity reference)

Plain gcc, -O2, OpenMP over independent output samples only.  Run as
`python -m oracle.build` or call build().
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "lisa_oracle.c")
LIBS = {
    "f64": (os.path.join(HERE, "liboracle_f64.so"), []),
    "f80": (os.path.join(HERE, "liboracle_f80.so"), ["-DORC_REAL_LD"]),
}


def build(force=False):
    import fcntl
    with open(os.path.join(HERE, ".build.lock"), "w") as lock:   # several processes may build at once
        fcntl.flock(lock, fcntl.LOCK_EX)
        for _, (out, defs) in LIBS.items():
            if (not force and os.path.exists(out)
                    and os.path.getmtime(out) >= os.path.getmtime(SRC)):
                continue
            # -ffp-contract=off: no fused multiply-adds the source does not spell out
            tmp = f"{out}.{os.getpid()}.tmp"
            cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-ffp-contract=off",
                   "-Wall", "-Wextra", *defs, "-o", tmp, SRC, "-lm"]
            subprocess.run(cmd, check=True)
            os.replace(tmp, out)
    return {k: v[0] for k, v in LIBS.items()}


if __name__ == "__main__":
    print(build(force=True))
