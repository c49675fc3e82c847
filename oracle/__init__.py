"""ORACLE package -- test infrastructure only (see mg.py header).  Never imported by the product path."""
from . import mg  # noqa: F401
