"""Write tests/golden/oracle_triples_<cfg>.txt: +T / (T) / -T of the CPU ORACLE (and nothing else).

    python tests/golden/make_oracle_triples.py cfg1

Calls only oracle/ and the shared input generator.  Amplitudes: ccsd_inputs.random_amplitudes(o, v, 35, 0.01)
(seeded, antisymmetric, CN(0, 0.01^2)); the energies are eqs 39, 41, 43 in reading G22.
"""
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import ccsd_inputs as ci  # noqa: E402
from oracle.ccsd_oracle import OracleCCSD, num_threads, unpack_t2  # noqa: E402
from oracle.triples_oracle import OracleTriples  # noqa: E402


def main():
    cfg = sys.argv[1]
    inp = ci.make_config(cfg)
    o, v = inp.nocc, inp.nvir
    t0 = time.time()
    oc = OracleCCSD(inp.h, inp.B, o, v, restricted=True)
    t1, t2p = ci.random_amplitudes(o, v, 35, 0.01)
    e = OracleTriples(oc, t1=t1, t2=unpack_t2(t2p, o, v)).energies(restricted=True)
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), f"oracle_triples_{cfg}.txt")
    with open(path, "w") as fh:
        fh.write(f"# oracle triples corrections, {cfg}: nocc={o} nvir={v} naux={inp.naux} seed={inp.seed}; amplitudes "
                 "random_amplitudes(o, v, 35, 0.01)\n")
        fh.write("# written by tests/golden/make_oracle_triples.py (oracle/ only, i<j<k restricted sum); "
                 f"host threads {num_threads()}, {time.time() - t0:.0f} s\n# key  Re(E)  Im(E)\n")
        for key in ("+T", "(T)", "-T"):
            fh.write(f"{key} {e[key].real!r} {e[key].imag!r}\n")
            print(key, e[key])


if __name__ == "__main__":
    main()
