"""Prints the oracle's own values for the rows of tests/golden/*.txt so that a reader can diff them against the
cited sources.  Calls only oracle/ (never the CUDA path).  The committed fixtures hold the CITED values
(SURVEY.md probes / published known answers), not this script's output."""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import oracle as O  # noqa: E402

if __name__ == "__main__":
    print("# philox"); print(" ".join("%08x" % x for x in O.philox4x32_10((0, 0, 0, 0), (0, 0))))
    print("# thermal cfg1"); print(O.thermal(300, 870, O.MUB, 1.25e-25, 8e5))
    print("# newell (3,2,1) unit cubes"); print(O.newell(3, 2, 1, 1, 1, 1))
