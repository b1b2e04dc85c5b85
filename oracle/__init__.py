"""CPU oracle package — TEST INFRASTRUCTURE ONLY (see uf_oracle.py header)."""
from .uf_oracle import UFOracle  # noqa: F401
