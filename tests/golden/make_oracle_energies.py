"""Write tests/golden/oracle_lockstep_<cfg>.txt: lock-step energies of the CPU ORACLE (and nothing else).

    python tests/golden/make_oracle_energies.py cfg2 10 [output file]

Calls only oracle/ and the shared input generator.  The file lists E (Re, Im) and ||S/D||_2 of the MP2 start and of
every iteration with DIIS(6) (reading G13), to be compared with the CUDA library's ccsd_iterate by the GPU tests.
The wall seconds of every REAL oracle iteration are appended to tests/golden/oracle_iteration_seconds.txt (the
genuine full-iteration CPU times bench.py quotes beside its slab-scaled cpu_baseline numbers).
"""
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import ccsd_inputs as ci  # noqa: E402
from oracle.ccsd_oracle import OracleCCSD, num_threads  # noqa: E402


def main():
    cfg = sys.argv[1]
    niter = int(sys.argv[2])
    inp = ci.make_config(cfg)
    t0 = time.time()
    oc = OracleCCSD(inp.h, inp.B, inp.nocc, inp.nvir, ndiis=6, restricted=True)
    lines = [f"# oracle lock-step energies, {cfg}: nocc={inp.nocc} nvir={inp.nvir} naux={inp.naux} seed={inp.seed}",
             "# written by tests/golden/make_oracle_energies.py (oracle/ only, restricted-sum mode, DIIS(6))",
             f"# host threads: {num_threads()}",
             "# iteration  Re(E)  Im(E)  ||S/D||_2 of the residual evaluated in that iteration (nan for the MP2 start)"]
    path = sys.argv[3] if len(sys.argv) > 3 else \
        os.path.join(os.path.dirname(os.path.abspath(__file__)), f"oracle_lockstep_{cfg}.txt")

    def flush():   # rewritten after every iteration: a long run that is cut short still leaves its finished lines
        with open(path, "w") as fh:
            fh.write("\n".join(lines) + "\n")

    e = oc.energy()
    lines.append(f"0 {e.real!r} {e.imag!r} nan")
    print(lines[-1], f"(setup {time.time() - t0:.0f} s)", flush=True)
    flush()
    setup_s = time.time() - t0
    secs = []
    for it in range(1, niter + 1):
        t1 = time.time()
        e, sn = oc.iterate()
        secs.append(time.time() - t1)
        lines.append(f"{it} {e.real!r} {e.imag!r} {sn!r}")
        print(lines[-1], f"({secs[-1]:.0f} s)", flush=True)
        flush()
    if secs:
        rec = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_iteration_seconds.txt")
        new = not os.path.exists(rec)
        with open(rec, "a") as fh:
            if new:
                fh.write("# wall seconds of real full oracle iterations (OracleCCSD.iterate, restricted-sum mode), written by\n"
                         "# tests/golden/make_oracle_energies.py; columns: config  host_threads  iterations  median_seconds_per_iteration"
                         "  setup_seconds(Fock + six integral classes)  host\n")
            fh.write(f"{cfg} {num_threads()} {len(secs)} {sorted(secs)[len(secs) // 2]:.1f} {setup_s:.1f} {os.uname().nodename}\n")


if __name__ == "__main__":
    main()
