"""CPU oracle (test infrastructure). See cs_oracle.cpp / cs_oracle.py. Never imported by the CUDA path."""
