import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200, sm_100a); run with -m gpu")


def pytest_collection_modifyitems(config, items):
    # GPU tests are selected with -m gpu; when they are selected on a box without a device they
    # must FAIL loudly (no silent skip, no CPU fallback), so nothing is auto-skipped here.
    return


class _NbDebug:
    """The library's debugging switches (include/nb_debug.h) with monkeypatch's setenv / delenv shape: every switch a
    test sets is restored to its default when the test ends.  The library reads no environment variable after start."""

    def __init__(self):
        self._touched = set()

    def setenv(self, key, value):
        import paper_astro_ph_0703100_b200 as nb
        nb.debug_set(key, str(value))
        self._touched.add(key)

    def delenv(self, key, raising=True):
        import paper_astro_ph_0703100_b200 as nb
        nb.debug_set(key, None)

    def restore(self):
        import paper_astro_ph_0703100_b200 as nb
        for key in self._touched:
            nb.debug_set(key, None)
        self._touched.clear()


@pytest.fixture
def nbdebug():
    d = _NbDebug()
    yield d
    d.restore()
