"""Test-side alias of oracle/batch.py (the oracle over all (b, h) units of a synthetic Workload)."""
from oracle.batch import OracleBatch  # noqa: F401
