"""Build the C oracle (TEST INFRASTRUCTURE, not product code).

`python -m oracle.build` or `oracle.build.build()` compiles
oracle/attention_oracle.c into oracle/liboracle_attn.so with
`gcc -O2 -ffp-contract=off -fopenmp` (the oracle is timed as it
stands, never tuned).  Building the checker is not using it: __graft_entry__.build()
calls this, the product path never loads the result.
"""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_HERE, "attention_oracle.c")
LIB = os.path.join(_HERE, "liboracle_attn.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
           "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
