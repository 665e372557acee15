"""python -m oracle : (re)build liboracle.so from oracle.cpp."""
from . import build

print(build(force=True))
