"""-m "not gpu": the C-ABI library loads here and exports every symbol include/nb.h declares; the
argument checks that need no device answer as the header says.  No compute calls."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def nbmod():
    import __graft_entry__ as g
    g.build()
    import paper_1409_5474_b200 as nbm
    return nbm


def _declared():
    with open(os.path.join(ROOT, "include", "nb.h")) as f:
        text = re.sub(r"/\*.*?\*/", "", f.read(), flags=re.S)
    return sorted(set(re.findall(r"\b(nb_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_exported(nbmod):
    names = _declared()
    assert len(names) >= 20
    lib = ctypes.CDLL(nbmod.binding.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), n
    # the binding lists the same names, and wraps each of them
    assert sorted(nbmod.binding.EXPORTS) == names
    for n in names:
        assert callable(getattr(nbmod.binding, n)), n


def test_no_torch_types_in_signatures():
    with open(os.path.join(ROOT, "include", "nb.h")) as f:
        text = f.read()
    assert "torch" not in text and "at::" not in text and "#include <cuda" not in text
    assert 'extern "C"' in text


def test_host_side_answers(nbmod):
    nb = nbmod.binding
    assert nb.nb_version().startswith("nb ")
    assert nb.nb_strerror(nb.NB_OK) == "ok"
    for s in (nb.NB_ERR_ARG, nb.NB_ERR_ALLOC, nb.NB_ERR_CUDA, nb.NB_ERR_INDEX, nb.NB_ERR_STATE,
              nb.NB_ERR_ARCH):
        assert nb.nb_strerror(s) not in ("ok", "unknown status")
    assert nb.nb_strerror(-99) == "unknown status"
    # workspace size: monotone, covers at least store (112 B) + pack (44 B) per particle
    w1, w2 = nb.nb_workspace_bytes(1 << 16, 1 << 16), nb.nb_workspace_bytes(1 << 20, 1 << 20)
    assert w2 > w1 >= (1 << 16) * (112 + 44)
    assert w2 % 256 == 0
    assert nb.nb_workspace_bytes(-1, 1) == 0


def test_create_fails_loudly_without_a_b200(nbmod):
    """No CPU fallback: on a box without a compute-capability-10.x GPU nb_create is an error."""
    torch = pytest.importorskip("torch")
    if torch.cuda.is_available() and torch.cuda.get_device_capability(0)[0] == 10:
        pytest.skip("a B200 is present")
    nb = nbmod.binding
    with pytest.raises(nb.NBError) as e:
        nb.nb_create(16, 16, 0, None)
    assert e.value.status in (nb.NB_ERR_CUDA, nb.NB_ERR_ARCH)
    with pytest.raises(nb.NBError):
        nb.nb_create(0, 16, 0, None)
