"""Test helper for the local / non-local split: the atom reordering lives with the generators."""
from paper_2006_09167_b200.workloads import local_first  # noqa: F401
