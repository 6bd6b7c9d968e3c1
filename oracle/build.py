"""Build step for the CPU oracle: `python oracle/build.py` -> oracle/libgwmf_oracle.so (gcc)."""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

if __name__ == "__main__":
    import oracle
    print(oracle.build(force=True))
