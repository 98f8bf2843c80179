"""QTAM forward / inverse Q-transform on B200 (sm_100a): thin ctypes binding over libqtam.so.

Importing the package is cheap; the CUDA library is loaded on first use (see .binding).
"""
__all__ = ["binding", "inputs"]
