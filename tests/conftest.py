import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HERE = os.path.dirname(os.path.abspath(__file__))
for _p in (ROOT, HERE):
    if _p not in sys.path:
        sys.path.insert(0, _p)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (runs on the B200 box)")
    # a checkout without built artefacts (they are git-ignored): compile the product library and the oracle once.
    # Building is not a fallback: a missing or failed build still makes every test that needs the library fail.
    try:
        from paper_2606_30391_b200.build import LIB, build as build_lib
        if not os.path.exists(LIB):
            build_lib()
    except Exception as e:                              # noqa: BLE001 - reported by the tests that need the library
        print(f"conftest: could not build libfestina_eval.so: {e}", file=sys.stderr)
    try:
        from oracle.build import build as build_oracle
        build_oracle()
    except Exception as e:                              # noqa: BLE001
        print(f"conftest: could not build the oracle: {e}", file=sys.stderr)


@pytest.fixture(scope="session")
def fs():
    """The CUDA library binding (only for -m gpu tests)."""
    import paper_2606_30391_b200 as pkg
    return pkg
